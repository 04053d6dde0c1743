// nmf_fused.cu -- placeholder until the fused per-pixel-tile kernel lands.
#include "nmf_common.cuh"
void   nmf_fused_configure(nmf_plan* p) { p->f_kp = 0; p->f_ctas = 0; }
size_t nmf_fused_workspace(const nmf_plan*) { return 0; }
bool   nmf_fused_available(const nmf_plan*) { return false; }
int    nmf_fused_fit(nmf_plan*, const float*, const float*, float*, float*, int, int) { return NMF_ERR_UNSUPPORTED; }
