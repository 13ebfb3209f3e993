// mk_syn_gemm.cu — synthesis contraction for large focal batches (compute-bound regime):
// per bin k a dense complex GEMM   S^_k[r][f] = sum_s R^_k[r][s] * N^_k[s][f],  M = nrec, K = nshot, N = nfoc,
// batched over the nb bins of the band (eq. (1); BASELINE.json north_star (b)).
// FP32 FFMA path: 128 x 64 complex CTA tile, 8 x 4 complex register tile per thread (4 FFMA per complex MAC),
// operands staged by a 3-stage cp.async pipeline in their natural layouts (A rows = shots fastest, B rows = focal
// points fastest), so no transposition and no split of re/im is needed.  Exact fp32 accumulate (no TF32).
#include "mk_internal.cuh"

namespace mk {

namespace {

constexpr int BM = 128, BN = 64, BK = 16, STAGES = 3;
constexpr int AST = BK + 2;  // padded A row (complex): 144 B keeps LDS.128 conflict-free across 8 consecutive rows
constexpr int kThreads = 256;
constexpr int TM = 8, TN = 4;
constexpr size_t kSmemA = (size_t)STAGES * BM * AST * sizeof(float2);
constexpr size_t kSmemB = (size_t)STAGES * BK * BN * sizeof(float2);

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool pred) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  const int sz = pred ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

// grid (ceil(ldf/BN), ceil(n/BM), nb).  A = Rhat [n][nb][ld], B = Nhat [nb][ld][ldf], C = Shat [n][nb][ldf]
__global__ void __launch_bounds__(kThreads, 2) k_syn_gemm_ffma(const float2* __restrict__ Rhat, const float2* __restrict__ Nhat,
                                                               float2* __restrict__ Shat, int n, int nb, int ld, int ldf) {
  extern __shared__ float4 smem4[];
  float2* sA = reinterpret_cast<float2*>(smem4);                                        // [STAGES][BM][AST]
  float2* sB = reinterpret_cast<float2*>(reinterpret_cast<char*>(smem4) + kSmemA);      // [STAGES][BK][BN]
  const int kk = blockIdx.z, m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ty = (warp >> 2) * 8 + (lane >> 2);  // 0..15 : rows ty + 16 i
  const int tx = (warp & 3) * 4 + (lane & 3);    // 0..15 : cols 4 tx .. 4 tx + 3
  const size_t lda = (size_t)nb * ld;
  const float2* Ag = Rhat + (size_t)kk * ld;
  const float2* Bg = Nhat + (size_t)kk * ld * ldf;
  const int KT = ld / BK;

  auto load_tile = [&](int kt, int st) {
    const int k0 = kt * BK;
#pragma unroll
    for (int i = 0; i < (BM * BK / 2) / kThreads; ++i) {  // 4 x 16-byte chunks of A
      const int cidx = tid + i * kThreads;
      const int row = cidx >> 3, c2 = (cidx & 7) * 2;
      const bool ok = (m0 + row) < n;
      const float2* src = Ag + (size_t)(ok ? m0 + row : 0) * lda + k0 + c2;
      cp_async16(sA + ((size_t)st * BM + row) * AST + c2, src, ok);
    }
#pragma unroll
    for (int i = 0; i < (BK * BN / 2) / kThreads; ++i) {  // 2 x 16-byte chunks of B
      const int cidx = tid + i * kThreads;
      const int row = cidx >> 5, c2 = (cidx & 31) * 2;
      const bool ok = (n0 + c2) < ldf;
      const float2* src = Bg + (size_t)(k0 + row) * ldf + (ok ? n0 + c2 : 0);
      cp_async16(sB + ((size_t)st * BK + row) * BN + c2, src, ok);
    }
  };

  float2 acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = make_float2(0.f, 0.f);

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KT) load_tile(s, s);
    cp_async_commit();
  }
  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      const int nk = kt + STAGES - 1;
      if (nk < KT) load_tile(nk, nk % STAGES);
      cp_async_commit();
    }
    const int st = kt % STAGES;
    const float2* a_base = sA + ((size_t)st * BM + ty) * AST;
    const float2* b_base = sB + (size_t)st * BK * BN + tx * TN;
#pragma unroll
    for (int k2 = 0; k2 < BK; k2 += 2) {
      float4 a[TM];
#pragma unroll
      for (int i = 0; i < TM; ++i) a[i] = *reinterpret_cast<const float4*>(a_base + (size_t)i * 16 * AST + k2);
      float4 b0[TN / 2], b1[TN / 2];
#pragma unroll
      for (int q = 0; q < TN / 2; ++q) {
        b0[q] = *reinterpret_cast<const float4*>(b_base + (size_t)k2 * BN + 2 * q);
        b1[q] = *reinterpret_cast<const float4*>(b_base + (size_t)(k2 + 1) * BN + 2 * q);
      }
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int q = 0; q < TN / 2; ++q) {
          // s = k2: a = (x + i y), b = b0 ; s = k2+1: a = (z + i w), b = b1
          float2& c0 = acc[i][2 * q];
          float2& c1 = acc[i][2 * q + 1];
          c0.x = fmaf(a[i].x, b0[q].x, c0.x);
          c0.y = fmaf(a[i].x, b0[q].y, c0.y);
          c1.x = fmaf(a[i].x, b0[q].z, c1.x);
          c1.y = fmaf(a[i].x, b0[q].w, c1.y);
          c0.x = fmaf(-a[i].y, b0[q].y, c0.x);
          c0.y = fmaf(a[i].y, b0[q].x, c0.y);
          c1.x = fmaf(-a[i].y, b0[q].w, c1.x);
          c1.y = fmaf(a[i].y, b0[q].z, c1.y);
          c0.x = fmaf(a[i].z, b1[q].x, c0.x);
          c0.y = fmaf(a[i].z, b1[q].y, c0.y);
          c1.x = fmaf(a[i].z, b1[q].z, c1.x);
          c1.y = fmaf(a[i].z, b1[q].w, c1.y);
          c0.x = fmaf(-a[i].w, b1[q].y, c0.x);
          c0.y = fmaf(a[i].w, b1[q].x, c0.y);
          c1.x = fmaf(-a[i].w, b1[q].w, c1.x);
          c1.y = fmaf(a[i].w, b1[q].z, c1.y);
        }
    }
  }
  cp_async_wait<0>();
  // epilogue
  const int col = n0 + tx * TN;
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int r = m0 + ty + 16 * i;
    if (r >= n) continue;
    float2* dst = Shat + ((size_t)r * nb + kk) * ldf + col;
#pragma unroll
    for (int q = 0; q < TN / 2; ++q)
      if (col + 2 * q < ldf)
        *reinterpret_cast<float4*>(dst + 2 * q) = make_float4(acc[i][2 * q].x, acc[i][2 * q].y, acc[i][2 * q + 1].x, acc[i][2 * q + 1].y);
  }
}

}  // namespace

int launch_syn_gemm(mk_ctx* c, const RowBlock& rb, const float2* d_Nhat, float2* d_Shat, int ldf) {
  const size_t smem = kSmemA + kSmemB;
  if (int rc = check_cuda(c, cudaFuncSetAttribute(k_syn_gemm_ffma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                          "cudaFuncSetAttribute"))
    return rc;
  // the block holds the rows r0 .. r0 + nrow - 1 of R^; S^ is indexed by the global receiver
  const dim3 grid((ldf + BN - 1) / BN, (rb.nrow + BM - 1) / BM, c->nb);
  k_syn_gemm_ffma<<<grid, kThreads, smem, c->stream>>>(rb.Rhat, d_Nhat, d_Shat + (size_t)rb.r0 * c->nb * ldf, rb.nrow, c->nb, c->ld, ldf);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_syn_gemm_ffma");
}

}  // namespace mk
