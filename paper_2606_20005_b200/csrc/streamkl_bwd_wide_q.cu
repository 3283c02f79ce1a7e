// streamkl_bwd_wide_q.cu -- Q-owner instantiations of the wide-head-dim backward kernel (dQ1, dQ2).
#define SKL_OWNER_K 0
#include <algorithm>
#include "streamkl_bwd_wide.inc"
