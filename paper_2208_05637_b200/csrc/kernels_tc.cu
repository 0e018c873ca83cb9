// Tensor-core (tcgen05 / TMEM / TMA) path — placeholder until the fused kernel lands.
#include "nqs_internal.h"
bool tc_supported(const nqs_made *) { return false; }
int  tc_pack_upload(const nqs_made *) { return NQS_OK; }
void tc_pack_free(const nqs_made *) {}
int  launch_logpsi_tc(const nqs_made *, const ulonglong2 *, long long, float2 *, cudaStream_t) { return NQS_EUNSUPPORTED; }
int  launch_eloc_tc(const HamDev &, const nqs_made *, const ulonglong2 *, const float2 *, long long, float2 *, unsigned *, cudaStream_t) { return NQS_EUNSUPPORTED; }
size_t eloc_tc_ws_bytes(long long, const HamDev &) { return 0; }
