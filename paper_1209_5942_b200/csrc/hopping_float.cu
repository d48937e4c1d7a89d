// hopping_float.cu -- the single-precision instantiations of the hopping kernel (hopping.cu compiled a second time,
// see the note above launch_hopping_float there), a translation unit of its own so that it builds beside the
// double-precision half.
#define LQCD_HOP_FLOAT_PART
#include "hopping.cu"
