// streamkl_bwd_k.cu -- K-owner instantiations of the tcgen05 backward kernel (dK1, dK2).
#define SKL_OWNER_K 1
#include "streamkl_bwd_owner.inc"
