// (kind, n) pairs the SWAR kernel is compiled for: X(kind, n).  One object file per entry
// (build.py compiles swar_inst.cu once per entry with -DPAIRINGS_SWAR_KIND / -DPAIRINGS_SWAR_N).
// Values of n where pairings exist, from the smallest the kernel supports (n-2 >= 4) to the
// largest the paper computed (Tables 4/5: S(28), S(29), L(27), L(28)).
// unrolled inner Gray bits of the SWAR kernel (smallest gray_bits it accepts)
#define PAIRINGS_SWAR_H 5
#ifndef PAIRINGS_SWAR_LIST
#define PAIRINGS_SWAR_LIST(X) \
    X(0, 8) X(0, 9) X(0, 12) X(0, 13) X(0, 16) X(0, 17) X(0, 20) X(0, 21) X(0, 24) X(0, 25) X(0, 28) X(0, 29) \
    X(1, 7) X(1, 8) X(1, 11) X(1, 12) X(1, 15) X(1, 16) X(1, 19) X(1, 20) X(1, 23) X(1, 24) X(1, 27) X(1, 28)
#endif
