// s2_force_fp64_bank1.cu -- second instance of the uniform-operand sweep (s2_force_fp64.cu, "uniform-operand sweep"):
// a translation unit is a CUDA module with its own 64 KB constant bank, so compiling the bank kernels a second time
// gives the sweep a second j-bank to alternate with (the refill of one overlaps the sweep of the other).
#define S2_BANK_ONLY
#define S2_BANK_ID 1
#include "s2_force_fp64.cu"
