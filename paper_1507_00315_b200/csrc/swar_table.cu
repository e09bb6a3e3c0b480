// Table of the compiled SWAR specialisations (swar_list.h).
#include "internal.h"
#include "swar_list.h"

namespace pairings {

#define PAIRINGS_DECL(k, n) int swar_launch_##k##_##n(const KernelParams&, int, unsigned, void*);
PAIRINGS_SWAR_LIST(PAIRINGS_DECL)
#undef PAIRINGS_DECL

swar_launch_fn swar_lookup(int kind, int n) {
#define PAIRINGS_CASE(k, nn) if (kind == k && n == nn) return &swar_launch_##k##_##nn;
    PAIRINGS_SWAR_LIST(PAIRINGS_CASE)
#undef PAIRINGS_CASE
    return nullptr;
}

int swar_min_gray_bits() { return PAIRINGS_SWAR_H; }

const char* swar_list() {
#define PAIRINGS_STR(k, nn) #k ":" #nn " "
    return PAIRINGS_SWAR_LIST(PAIRINGS_STR);
#undef PAIRINGS_STR
}

}  // namespace pairings
