"""Writes rope_d2_closed_form.txt from the closed form of Eq. 2 at D = 2.

score(t, j) = (R_t q) . (R_j k) / sqrt(2) = |q||k| cos((p_j - p_t) + arg(k) - arg(q)) / sqrt(2)
because D = 2 has the single frequency f_0 = theta^0 = 1.  Uses only `math`.
"""
import math
import os

ROWS = [  # p_t, p_j, q, k
    (0, 0, (1.0, 0.0), (1.0, 0.0)),
    (1, 0, (1.0, 0.0), (1.0, 0.0)),
    (3, 1, (1.0, 0.0), (1.0, 0.0)),
    (3, 1, (0.0, 1.0), (1.0, 0.0)),
    (7, 2, (0.5, -1.5), (2.0, 0.25)),
    (4099, 4096, (1.0, 1.0), (-1.0, 2.0)),
    (1000003, 1000000, (1.0, 1.0), (-1.0, 2.0)),
]

if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "rope_d2_closed_form.txt"), "w") as f:
        f.write("# p_t p_j q0 q1 k0 k1 score   (Eq. 2, PAPER.md:102, D=2 closed form; see README.md)\n")
        for pt, pj, q, k in ROWS:
            ang = (pj - pt) + math.atan2(k[1], k[0]) - math.atan2(q[1], q[0])
            s = math.hypot(*q) * math.hypot(*k) * math.cos(ang) / math.sqrt(2.0)
            f.write(f"{pt} {pj} {q[0]!r} {q[1]!r} {k[0]!r} {k[1]!r} {s!r}\n")
