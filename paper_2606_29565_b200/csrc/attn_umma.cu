// attn_umma.cu -- tcgen05/TMEM kernel for a1 + a2 (placeholder until the UMMA path lands).
#include "common.cuh"

bool prepos_attn_umma_supported(const prepos_ctx *) { return false; }

int prepos_launch_attn_umma(prepos_ctx *, const AttnArgs &, int, cudaStream_t) { return PREPOS_E_SHAPE; }
