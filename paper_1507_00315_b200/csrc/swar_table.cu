// Table of compiled SWAR specialisations (filled in by swar_inst_*.cu).
#include "internal.h"

namespace pairings {
swar_launch_fn swar_lookup(int, int) { return nullptr; }
int swar_min_gray_bits() { return 4; }
const char* swar_list() { return "(none)"; }
}  // namespace pairings
