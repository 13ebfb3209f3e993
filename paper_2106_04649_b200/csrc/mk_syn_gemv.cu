// mk_syn_gemv.cu — synthesis contraction for few focal points (bandwidth-bound regime):
//   S^[r][k][f] = sum_s R^[r][k][s] * N^[k][s][f]          (dt * w[s] already folded into R^ at ingest)
// eq. (1) of the paper evaluated in the frequency domain.  The paper runs this as a pointwise
// multiply kernel that materialises d_RF followed by a CUB segmented reduction; here the
// product is never stored: every row of R^ (one receiver, one bin: ld complex, contiguous) is streamed from HBM
// exactly once with 128-bit loads, multiplied against the bin's N^ column block held in shared memory, and reduced
// with warp shuffles.  Algorithmic traffic: 8 bytes per complex element of R^.
#include "mk_internal.cuh"

namespace mk {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
// receivers per CTA (measured, config-1 step over three 40-step runs: 32 rows 3.440 / 3.465 / 3.486 ms, 64 rows 3.429 / 3.455 /
// 3.476, 128 rows 3.460 / 3.485 / 3.509)
#ifndef MK_GEMV_ROWS_PER_CTA
#define MK_GEMV_ROWS_PER_CTA 64
#endif
constexpr int kRowsPerCta = MK_GEMV_ROWS_PER_CTA;  // receivers per CTA
// Rows of R^ a warp streams at once (x reuse, independent load streams), unroll of the chunk loop (loads in flight per
// stream) and CTAs per SM.  Measured on B200, config 1 (nfoc = 1, 1.30 GB of R^): (4, 2, 3) 6.81 TB/s, (4, 1, 4) 7.00,
// (2, 4, 4) 7.03; a pure read of the same bytes peaks at 7.70 TB/s.  Larger NFOC: registers decide (accumulators =
// rows x NFOC complex), the x reads from shared memory are 2 NFOC / rows bytes per byte of R^.
template <int NFOC>
struct Tune {
  // measured per NFOC on config 1's R^ (us per launch): 188, 209, 211, 248, 270, 305, 360, 383 for NFOC = 1..8
  static constexpr int kRows = NFOC == 1 ? 2 : (NFOC == 2 ? 4 : (NFOC <= 6 ? 2 : 4));
  static constexpr int kUnroll = NFOC == 1 ? 4 : (NFOC <= 4 ? 2 : 1);
  static constexpr int kMinBlocks = NFOC == 1 ? 4 : (NFOC <= 4 ? 3 : 2);
};

struct f8 {
  float v[8];
};
// 256-bit streaming load (sm_100: LDG.E.256), L1 no-allocate, L2 evict-first: R^ is read exactly once per synthesis
__device__ __forceinline__ f8 ld_stream(const float* p) {
  f8 r;
  asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]), "=f"(r.v[4]), "=f"(r.v[5]), "=f"(r.v[6]), "=f"(r.v[7])
               : "l"(p));
  return r;
}

__device__ __forceinline__ void cfma(float2& acc, float ar, float ai, float2 b) {
  acc.x = fmaf(ar, b.x, acc.x);
  acc.x = fmaf(-ai, b.y, acc.x);
  acc.y = fmaf(ar, b.y, acc.y);
  acc.y = fmaf(ai, b.x, acc.y);
}

// grid (nb, ceil(n / kRowsPerCta)).  Rhat [n][nb][ld], Nhat [nb][ld][NFOC], Shat [n][nb][NFOC].
template <int NFOC>
__global__ void __launch_bounds__(kThreads, Tune<NFOC>::kMinBlocks) k_syn_gemv(const float2* __restrict__ Rhat, const float2* __restrict__ Nhat,
                                                       float2* __restrict__ Shat, int n, int nb, int ld, int early_pf) {
  extern __shared__ float4 smem4[];
  pdl_trigger();
  if ((int)(blockIdx.y * gridDim.x + blockIdx.x) < early_pf) {   // the CTAs of the first wave: the others start long after the wait
    // R^ never changes during a run: the head of the first rows of every warp starts its way from HBM to L2 while the kernel
    // in front (which produces N^) is still draining.  A cache hint only: nothing is read before the wait.
    const int w0 = blockIdx.y * kRowsPerCta + (threadIdx.x >> 5) * Tune<NFOC>::kRows;
#pragma unroll
    for (int i = 0; i < Tune<NFOC>::kRows; ++i) {
      const float2* rp = Rhat + ((size_t)min(w0 + i, n - 1) * nb + blockIdx.x) * ld;
      const int c = threadIdx.x & 31;   // 4 KB per row: what the first loads of the chunk loop ask for
      if (c < (ld >> 4)) asm volatile("prefetch.global.L2 [%0];" ::"l"(rp + 16 * c));
    }
  }
  pdl_wait();   // N^ is the output of the kernel in front (mk_internal.cuh: launch_pdl)
  // N^ bin column in shared memory.  A lane always reads the four shots 4c .. 4c+3 of its 256-bit chunk c, so the natural
  // [shot][focal] order puts the lanes 32 NFOC bytes apart: for NFOC = 4, 8 every lane of a warp hits the same banks
  // (measured: 436 / 778 us against 210 us at NFOC = 3).  NFOC >= 4 therefore keeps x as [focal][e][chunk]: the lanes of
  // one load are consecutive.
  float2* x = reinterpret_cast<float2*>(smem4);
  const int kk = blockIdx.x;
  const int r_begin = blockIdx.y * kRowsPerCta;
  const int r_end = min(r_begin + kRowsPerCta, n);
  const int nchunk = ld >> 2;  // 256-bit chunk = 4 complex (ld is a multiple of 16)
  constexpr bool kTransposed = NFOC >= 4;
  if (!kTransposed) {
    const float4* src = reinterpret_cast<const float4*>(Nhat + (size_t)kk * ld * NFOC);
    for (int i = threadIdx.x; i < ld * NFOC / 2; i += kThreads) smem4[i] = __ldg(src + i);
  } else {
    const float2* src = Nhat + (size_t)kk * ld * NFOC;
    for (int i = threadIdx.x; i < ld * NFOC; i += kThreads) {
      const int s = i / NFOC, f = i - s * NFOC;
      x[(f * 4 + (s & 3)) * nchunk + (s >> 2)] = __ldg(src + i);
    }
  }
  __syncthreads();
  constexpr int kRows = Tune<NFOC>::kRows;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int r0 = r_begin + warp * kRows; r0 < r_end; r0 += kWarps * kRows) {
    const float* row[kRows];
#pragma unroll
    for (int i = 0; i < kRows; ++i) {
      const int r = min(r0 + i, n - 1);
      row[i] = reinterpret_cast<const float*>(Rhat + ((size_t)r * nb + kk) * ld);
    }
    float2 acc[kRows][NFOC];
#pragma unroll
    for (int i = 0; i < kRows; ++i)
#pragma unroll
      for (int f = 0; f < NFOC; ++f) acc[i][f] = make_float2(0.f, 0.f);
#pragma unroll Tune<NFOC>::kUnroll
    for (int c = lane; c < nchunk; c += 32) {
      f8 a[kRows];
#pragma unroll
      for (int i = 0; i < kRows; ++i) a[i] = ld_stream(row[i] + 8 * c);
#pragma unroll
      for (int e = 0; e < 4; ++e)
#pragma unroll
        for (int f = 0; f < NFOC; ++f) {
          const float2 xv = kTransposed ? x[(f * 4 + e) * nchunk + c] : x[(4 * c + e) * NFOC + f];
#pragma unroll
          for (int i = 0; i < kRows; ++i) cfma(acc[i][f], a[i].v[2 * e], a[i].v[2 * e + 1], xv);
        }
    }
#pragma unroll
    for (int i = 0; i < kRows; ++i)
#pragma unroll
      for (int f = 0; f < NFOC; ++f) {
        float2 v = acc[i][f];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
          v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        }
        if (lane == 0 && r0 + i < r_end) Shat[((size_t)(r0 + i) * nb + kk) * NFOC + f] = v;
      }
  }
}

template <int NFOC>
int launch_t(mk_ctx* c, const RowBlock& rb, const float2* d_Nhat, float2* d_Shat) {
  const size_t smem = (size_t)c->ld * NFOC * sizeof(float2);
  auto kern = k_syn_gemv<NFOC>;
  if (int rc = check_cuda(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "cudaFuncSetAttribute"))
    return rc;
  // the block holds the rows r0 .. r0 + nrow - 1 of R^; S^ is indexed by the global receiver
  const dim3 grid(c->nb, (rb.nrow + kRowsPerCta - 1) / kRowsPerCta);
  if (int rc = check_cuda(c, launch_pdl(c, kern, grid, dim3(kThreads), smem, rb.Rhat, d_Nhat, d_Shat + (size_t)rb.r0 * c->nb * NFOC, rb.nrow, c->nb, c->ld, (c->tune & 8192) ? 0 : c->num_sms * Tune<NFOC>::kMinBlocks), "k_syn_gemv")) return rc;
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_syn_gemv");
}

}  // namespace

bool gemv_supported(const mk_ctx* c, int nfoc) {
  return nfoc >= 1 && nfoc <= 8 && (size_t)c->ld * nfoc * sizeof(float2) <= 96 * 1024;
}

int launch_syn_gemv(mk_ctx* c, const RowBlock& rb, const float2* d_Nhat, float2* d_Shat, int nfoc) {
  switch (nfoc) {
    case 1: return launch_t<1>(c, rb, d_Nhat, d_Shat);
    case 2: return launch_t<2>(c, rb, d_Nhat, d_Shat);
    case 3: return launch_t<3>(c, rb, d_Nhat, d_Shat);
    case 4: return launch_t<4>(c, rb, d_Nhat, d_Shat);
    case 5: return launch_t<5>(c, rb, d_Nhat, d_Shat);
    case 6: return launch_t<6>(c, rb, d_Nhat, d_Shat);
    case 7: return launch_t<7>(c, rb, d_Nhat, d_Shat);
    case 8: return launch_t<8>(c, rb, d_Nhat, d_Shat);
    default: return set_err(c, MK_ERR_INVALID_ARG, "gemv regime needs 1 <= nfoc <= 8");
  }
}

}  // namespace mk
