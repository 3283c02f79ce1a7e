// streamkl_bwd_wide_k.cu -- K-owner instantiations of the wide-head-dim backward kernel (dK1, dK2).
#define SKL_OWNER_K 1
#include <algorithm>
#include "streamkl_bwd_wide.inc"
