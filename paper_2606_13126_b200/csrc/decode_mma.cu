#include "internal.h"
namespace minipic {
bool decode_mma_supported(const Ctx&) { return false; }
void launch_decode_mma(const Ctx&, const DecodeArgs&, const SplitPlan&, float*, float*) {}
}  // namespace minipic
