#include "internal.h"
namespace minipic {
bool prefill_sm100_supported(const Ctx&) { return false; }
size_t prefill_sm100_workspace_bytes(const Ctx&, int, int) { return 0; }
bool launch_prefill_sm100(const Ctx&, const PrefillArgs&) { return false; }
}  // namespace minipic
