// mk_syn_gemv_q16.cu — NEXT-4: lossy-compressed R^ for the bandwidth-bound regime (nfoc <= 8).
// The paper's predecessor compressed R with ZFP to "accelerate data loading"; for one focal point the
// synthesis is a pure stream of R^ (§8(a) a2: 1 flop per byte), so the only lever left on a kernel that already reads at
// the HBM ceiling is fewer bytes.  Format "q16" (MK_OPT_RHAT_FORMAT = 1): block floating point, 16-bit mantissas —
//   a row R^[r][k][.] is cut into blocks of 16 shots; a block stores one fp32 scale  sc = max(|re|, |im|) / 32767  and,
//   per complex element, the two int16  q = rint(v / sc)  packed into one 32-bit word (re low, im high);
//   the value used is  q * sc:  absolute error <= sc / 2 = 1.5e-5 of the block's largest component, rms 8.8e-6.
// Bytes per complex element: 4 + 4/16 = 4.25 instead of 8.  Accumulation stays fp32 (integer mantissas are exact in
// fp32; a block's partial sum is scaled once).  The tolerance this path is held to is its own, not
// north_star's 2e-5: the compression error is a property of the format, not of the arithmetic.
#include "mk_internal.cuh"

namespace mk {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kRowsPerCta = 64;
constexpr int kQBlock = 16;  // shots per scale

template <int NFOC>
struct TuneQ {
  // a row of config 1 is 76 chunks: at most 3 per lane, so an unroll of 3 puts the whole row in flight
  static constexpr int kRows = 2;
  static constexpr int kUnroll = NFOC <= 2 ? 3 : (NFOC <= 4 ? 2 : 1);
  static constexpr int kMinBlocks = NFOC <= 2 ? 3 : 2;
};

struct u8x {
  uint32_t v[8];
};
__device__ __forceinline__ u8x ld_stream_u(const uint32_t* p) {
  u8x r;
  asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]), "=r"(r.v[7])
               : "l"(p));
  return r;
}

__device__ __forceinline__ void cfma(float2& acc, float ar, float ai, float2 b) {
  acc.x = fmaf(ar, b.x, acc.x);
  acc.x = fmaf(-ai, b.y, acc.x);
  acc.y = fmaf(ar, b.y, acc.y);
  acc.y = fmaf(ai, b.x, acc.y);
}

// grid (nb, ceil(n / kRowsPerCta)).  Rq [n][nb][ld] packed int16 pairs, Rsc [n][nb][ld / 16], Nhat [nb][ld][NFOC],
// Shat [n][nb][NFOC].  A lane streams 256-bit chunks of 8 complex elements; two neighbouring lanes share a scale.
template <int NFOC>
__global__ void __launch_bounds__(kThreads, TuneQ<NFOC>::kMinBlocks)
k_syn_gemv_q16(const uint32_t* __restrict__ Rq, const float* __restrict__ Rsc, const float2* __restrict__ Nhat, float2* __restrict__ Shat,
               int n, int nb, int ld) {
  extern __shared__ float4 smem4[];
  float2* x = reinterpret_cast<float2*>(smem4);
  const int kk = blockIdx.x;
  const int r_begin = blockIdx.y * kRowsPerCta;
  const int r_end = min(r_begin + kRowsPerCta, n);
  const int nchunk = ld >> 3;  // chunk = 8 complex = 32 bytes (ld is a multiple of 16)
  {  // N^ bin column as [focal][e][chunk]: the lanes of one read are consecutive (no bank conflicts for any NFOC)
    const float2* src = Nhat + (size_t)kk * ld * NFOC;
    for (int i = threadIdx.x; i < ld * NFOC; i += kThreads) {
      const int s = i / NFOC, f = i - s * NFOC;
      x[(f * 8 + (s & 7)) * nchunk + (s >> 3)] = __ldg(src + i);
    }
  }
  __syncthreads();
  constexpr int kRows = TuneQ<NFOC>::kRows;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int r0 = r_begin + warp * kRows; r0 < r_end; r0 += kWarps * kRows) {
    const uint32_t* row[kRows];
    const float* srow[kRows];
#pragma unroll
    for (int i = 0; i < kRows; ++i) {
      const int r = min(r0 + i, n - 1);
      row[i] = Rq + ((size_t)r * nb + kk) * ld;
      srow[i] = Rsc + ((size_t)r * nb + kk) * (ld / kQBlock);
    }
    float2 acc[kRows][NFOC];
#pragma unroll
    for (int i = 0; i < kRows; ++i)
#pragma unroll
      for (int f = 0; f < NFOC; ++f) acc[i][f] = make_float2(0.f, 0.f);
#pragma unroll TuneQ<NFOC>::kUnroll
    for (int c = lane; c < nchunk; c += 32) {
      u8x a[kRows];
      float sc[kRows];
#pragma unroll
      for (int i = 0; i < kRows; ++i) {
        a[i] = ld_stream_u(row[i] + 8 * c);
        sc[i] = __ldg(srow[i] + (c >> 1));
      }
      float2 part[kRows][NFOC];
#pragma unroll
      for (int i = 0; i < kRows; ++i)
#pragma unroll
        for (int f = 0; f < NFOC; ++f) part[i][f] = make_float2(0.f, 0.f);
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        float re[kRows], im[kRows];
#pragma unroll
        for (int i = 0; i < kRows; ++i) {
          const uint32_t w = a[i].v[e];
          re[i] = (float)(short)(w & 0xffffu);
          im[i] = (float)((int)w >> 16);
        }
#pragma unroll
        for (int f = 0; f < NFOC; ++f) {
          const float2 xv = x[(f * 8 + e) * nchunk + c];
#pragma unroll
          for (int i = 0; i < kRows; ++i) cfma(part[i][f], re[i], im[i], xv);
        }
      }
#pragma unroll
      for (int i = 0; i < kRows; ++i)
#pragma unroll
        for (int f = 0; f < NFOC; ++f) {
          acc[i][f].x = fmaf(sc[i], part[i][f].x, acc[i][f].x);
          acc[i][f].y = fmaf(sc[i], part[i][f].y, acc[i][f].y);
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

// Ingest: fp32 R^ of one sub-chunk of shots, stage [rows][ldc] (rows = n * nb; columns = shots of the sub-chunk, zero
// padded to a multiple of 16) -> packed mantissas and scales at columns shot0 .. of the rows of R^.  One thread per
// complex element, 16 lanes per block.
__global__ void k_quantize_q16(const float2* __restrict__ stage, uint32_t* __restrict__ Rq, float* __restrict__ Rsc, size_t rows, int ldc, int ld,
                               int shot0) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t row = idx / ldc;
  const int j = (int)(idx - row * ldc);
  const bool live = row < rows;
  const float2 v = live ? stage[row * ldc + j] : make_float2(0.f, 0.f);
  float m = fmaxf(fabsf(v.x), fabsf(v.y));
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (!live) return;
  const float sc = m / 32767.f, inv = m > 0.f ? 32767.f / m : 0.f;
  const int qr = max(-32767, min(32767, __float2int_rn(v.x * inv)));
  const int qi = max(-32767, min(32767, __float2int_rn(v.y * inv)));
  Rq[row * ld + shot0 + j] = ((uint32_t)qr & 0xffffu) | ((uint32_t)qi << 16);
  if ((j & (kQBlock - 1)) == 0) Rsc[row * (ld / kQBlock) + (shot0 + j) / kQBlock] = sc;
}

template <int NFOC>
int launch_t(mk_ctx* c, const float2* d_Nhat, float2* d_Shat) {
  const size_t smem = (size_t)c->ld * NFOC * sizeof(float2);
  auto kern = k_syn_gemv_q16<NFOC>;
  if (int rc = check_cuda(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "cudaFuncSetAttribute"))
    return rc;
  const dim3 grid(c->nb, (c->n + kRowsPerCta - 1) / kRowsPerCta);
  kern<<<grid, kThreads, smem, c->stream>>>(c->d_Rq, c->d_Rscale, d_Nhat, d_Shat, c->n, c->nb, c->ld);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_syn_gemv_q16");
}

}  // namespace

int launch_syn_gemv_q16(mk_ctx* c, const float2* d_Nhat, float2* d_Shat, int nfoc) {
  switch (nfoc) {
    case 1: return launch_t<1>(c, d_Nhat, d_Shat);
    case 2: return launch_t<2>(c, d_Nhat, d_Shat);
    case 3: return launch_t<3>(c, d_Nhat, d_Shat);
    case 4: return launch_t<4>(c, d_Nhat, d_Shat);
    case 5: return launch_t<5>(c, d_Nhat, d_Shat);
    case 6: return launch_t<6>(c, d_Nhat, d_Shat);
    case 7: return launch_t<7>(c, d_Nhat, d_Shat);
    case 8: return launch_t<8>(c, d_Nhat, d_Shat);
    default: return set_err(c, MK_ERR_INVALID_ARG, "compressed R^ (q16) serves the streaming regime only: 1 <= nfoc <= 8");
  }
}

int launch_quantize_q16(mk_ctx* c, const float2* d_stage, int ldc, int shot0) {
  const size_t rows = (size_t)c->n * c->nb, total = rows * ldc;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  k_quantize_q16<<<blocks, 256, 0, c->stream>>>(d_stage, c->d_Rq, c->d_Rscale, rows, ldc, c->ld, shot0);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_quantize_q16");
}

}  // namespace mk
