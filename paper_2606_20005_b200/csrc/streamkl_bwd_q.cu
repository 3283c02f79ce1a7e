// streamkl_bwd_q.cu -- Q-owner instantiations of the tcgen05 backward kernel (dQ1, dQ2) + the B1 pre-pass.
#define SKL_OWNER_K 0
#include "streamkl_bwd_owner.inc"
