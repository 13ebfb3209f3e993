// mk_fft_common.cuh — device helpers shared by the two transform paths (mk_fft_kernels.cu: generic shared-memory
// passes for any power-of-two nt; mk_fft_fast.cu: register-resident path for nt = 2048 / 4096).
#pragma once

#include "mk_internal.cuh"

namespace mk {

// a6 store: X = N^[k][r][f], into this rank's operand and, when peers are attached (row sharding), into theirs
__device__ __forceinline__ int operand_row(const OperandOut& O, int r) { return O.shot_of_rec ? __ldg(O.shot_of_rec + r) : r; }

__device__ __forceinline__ void store_operand(const OperandOut& O, int ld, int kk, int r, int f, float2 X) {
  const int s = operand_row(O, r);
  if (s < 0) return;
  const size_t idx = ((size_t)kk * ld + s) * O.ldf + f;
  O.plain[idx] = X;
  // compile-time indices: a run-time index into peer[] would make the compiler copy the whole struct to local memory
  // (measured: 155 local loads and generic-space stores in k_post_fast)
#pragma unroll
  for (int p = 0; p < kMaxPeers; ++p)
    if (p < O.npeer) O.peer[p][idx] = X;
}

// mk_fft_fast.cu: true when the register-resident path handles this context's nt (and it is not switched off)
bool fast_fft_ok(const mk_ctx* c);
int launch_load_R_fast(mk_ctx* c, const RowBlock& rb, const float* d_R_time, int shot0, int nshots);
int launch_fwd_fast(mk_ctx* c, const float* d_src, const OperandOut& O, int nfoc, bool conj_out, float* d_init_Tsrc);
int launch_inv_fast(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
                    const float* d_B, float sB);
int launch_post_fast(mk_ctx* c, const OperandOut& O, int parity_even, float* d_Ni_out);

}  // namespace mk
