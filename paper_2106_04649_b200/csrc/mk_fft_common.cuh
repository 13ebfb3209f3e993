// mk_fft_common.cuh — device helpers shared by the two transform paths (mk_fft_kernels.cu: generic shared-memory
// passes for any power-of-two nt; mk_fft_fast.cu: register-resident path for nt = 2048 / 4096).
#pragma once

#include "mk_internal.cuh"

namespace mk {

__device__ __forceinline__ float tf32_rna(float v) {
  unsigned u;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(v));
  return __uint_as_float(u);
}

// a6 store: X = N^[k][r][f] in the layout the contraction of the active regime reads, into this rank's operand and,
// when peers are attached (row sharding), into theirs
__device__ __forceinline__ void store_split_rows(float* hi, float* lo, size_t row0, int ldb, float2 X) {
  // regime 3 (mk_syn_tc.cu): real operand B' [nb][2 ld][ldb], rows (2r, 2r+1) = (X, iX) as interleaved floats,
  // split into a tf32 "hi" plane and a tf32 "lo" plane (3xTF32).
  const float hx = tf32_rna(X.x), hy = tf32_rna(X.y);
  const float lx = tf32_rna(X.x - hx), ly = tf32_rna(X.y - hy);
  *reinterpret_cast<float2*>(hi + row0) = make_float2(hx, hy);
  *reinterpret_cast<float2*>(hi + row0 + ldb) = make_float2(-hy, hx);
  *reinterpret_cast<float2*>(lo + row0) = make_float2(lx, ly);
  *reinterpret_cast<float2*>(lo + row0 + ldb) = make_float2(-ly, lx);
}

__device__ __forceinline__ void store_operand(const OperandOut& O, int ld, int kk, int r, int f, float2 X) {
  if (O.bhi == nullptr) {
    const size_t idx = ((size_t)kk * ld + r) * O.ldf + f;
    O.plain[idx] = X;
    for (int p = 0; p < O.npeer; ++p) reinterpret_cast<float2*>(O.peer[p][0])[idx] = X;
    return;
  }
  const size_t row0 = ((size_t)kk * 2 * ld + 2 * r) * O.ldb + 2 * f;
  store_split_rows(O.bhi, O.blo, row0, O.ldb, X);
  for (int p = 0; p < O.npeer; ++p) store_split_rows(O.peer[p][0], O.peer[p][1], row0, O.ldb, X);
}

// mk_fft_fast.cu: true when the register-resident path handles this context's nt (and it is not switched off)
bool fast_fft_ok(const mk_ctx* c);
int launch_load_R_fast(mk_ctx* c, const float* d_R_time, int shot0, int nshots);
int launch_fwd_fast(mk_ctx* c, const float* d_src, const OperandOut& O, int nfoc, bool conj_out, float* d_init_Tsrc);
int launch_inv_fast(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
                    const float* d_B, float sB);
int launch_post_fast(mk_ctx* c, const OperandOut& O, int parity_even, float* d_Ni_out);

}  // namespace mk
