// mk_syn_tc.cu — synthesis contraction for large focal batches on the 5th-generation tensor cores (SURVEY.md §8(f)
// NEXT-2; BASELINE.json north_star (b): "a tcgen05/TMEM 3xTF32 split path only if it meets the FP32 tolerance").
//
// Per bin k the complex GEMM  S^_k[r][f] = sum_s R^_k[r][s] N^_k[s][f]  (eq. (1)) is run as the REAL GEMM
//     C'[r][2f+c] = sum_{k'} A'[r][k'] B'[k'][2f+c],     k' = 2s + (0: re, 1: im),  c = (0: re, 1: im)
//   A'  = the row R^[r][k][.] read as 2 ld interleaved floats — R^ exactly as it sits in HBM (K-major, TMA, no copy);
//   B'  = rows (2s, 2s+1) = (N^[k][s][.], i N^[k][s][.]) as interleaved floats, written by the forward-transform
//         kernels (mk_fft_kernels.cu store_operand) already split into two tf32 planes  B' = Bhi + Blo;
//   C'  = S^[r][k][.] as interleaved floats — the layout k_post reads.
// 3xTF32: A' = Ahi + Alo with Ahi = the tf32 the tensor core sees when it reads the fp32 word (the low 13 mantissa
// bits are not used) and Alo = A' - Ahi (exact in fp32, computed on the fly by four "split" warps into a second
// shared-memory tile); every k'-chunk issues  Alo*Bhi + Ahi*Blo + Ahi*Bhi  into one fp32 accumulator in TMEM.  The dropped
// term Alo*Blo is O(2^-20) relative.
//
// Accumulation.  The tensor core adds into its fp32 accumulator with TRUNCATION, not round-to-nearest: measured on B200
// with one accumulator over the whole K extent the relative error of S^ grows linearly with the number of MMA steps
// (about 2e-8 per step: 6.8e-7 at n = 32, 2.9e-5 at n = 2048, against 1.2e-6 for the FFMA kernel), which breaks the
// 2e-5 per-iteration tolerance from n ~ 600 on.  So K is cut into CHUNKS of kChunkKb k'-blocks (24 MMA steps): every
// chunk starts a fresh TMEM accumulator, and the epilogue warps add the finished chunk into fp32 registers
// (round-to-nearest) while the tensor core works on the next chunk in the other TMEM buffer.  The error is then that
// of one chunk (~5e-7), independent of n.
//
// Kernel: persistent, one CTA per SM, warp-specialised, 384 threads —
//   warp 0      TMA producer: A' tile [128 rows][16 floats] (SWIZZLE_64B, K-major) and the two B' tiles
//               [16 k'][256 floats] (SWIZZLE_128B with 32-byte atoms, MN-major) per stage, 4 stages, mbarrier full/empty ring
//   warp 1      tcgen05.mma issuer (one thread): kind::tf32, M = 128, N <= 256, K = 8; chunk accumulators double-buffered
//               in TMEM (2 x 256 columns); tcgen05.commit releases the stage / publishes the chunk
//   warps 2-3   split warps: Alo tile of the stage
//   warps 4-11  epilogue: warp w owns TMEM lanes 32 (w % 4) .. +31 and the column half (w - 4) / 4; per chunk
//               tcgen05.ld 32x32b -> += 128 running sums in registers; per tile 128-bit global stores of S^
#include <cuda.h>

#include <algorithm>
#include <cstdlib>

#include "mk_internal.cuh"

namespace mk {

namespace {

constexpr int BM = 128;        // rows (receivers) per tile = TMEM lanes
constexpr int BN = 256;        // real columns (2 per focal point) per tile = TMEM columns per accumulator
constexpr int BK = 16;         // k' (floats of the interleaved shot dimension) per stage: 64-byte rows of A'
constexpr int UK = 8;          // k' per tcgen05.mma (kind::tf32)
constexpr int kMaxStages = 12;  // the ring has as many stages as fit (4 at N = 256, 11 for a single column block)
constexpr int kThreads = 384;  // 12 warps
constexpr int kChunkKb = 4;    // k'-blocks per accumulation chunk (24 MMA steps)
constexpr int kEpiWarps = 8;
constexpr uint32_t A_BYTES = BM * BK * 4;   // 8 KB
constexpr uint32_t BLK_BYTES = BK * 32 * 4;  // one 32-column block of a B' tile: 2 KB
// A stage = A raw, A lo (8 KB each), B hi, B lo (nblk column blocks each, nblk = min(8, ceil(columns / 32))): narrow
// focal batches move and hold only the columns they have, and get a deeper ring for it (HBM-bound regime)
// mp = M tiles (of 128 receivers) that share the stage's B' tile: 2 when the focal batch fits 128 columns, so that a
// stage feeds as many MMA cycles as a 256-column one with 32 KB instead of 2 x 24 KB of loads (the kernel is feed-bound)
__host__ __device__ constexpr uint32_t stage_bytes(int nblk, int mp) { return 2 * (uint32_t)mp * A_BYTES + 2 * (uint32_t)nblk * BLK_BYTES; }
constexpr size_t kSmemExtra = 1024 /*alignment slack*/ + 512 /*barriers*/;
constexpr uint32_t kTmemCols = 512;

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Bounded wait: a protocol bug traps (the launch fails with an error) instead of hanging the GPU.  The budget is a
// compile-time option: MK_MBAR_TIMEOUT_CYCLES (default 4e10 SM cycles, about 20 s — no stage of a healthy launch waits
// that long, not even under a profiler's replay or on a contended GPU); -DMK_MBAR_TIMEOUT_CYCLES=0 compiles the
// check out.
#ifndef MK_MBAR_TIMEOUT_CYCLES
#define MK_MBAR_TIMEOUT_CYCLES 40000000000LL
#endif
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
#if MK_MBAR_TIMEOUT_CYCLES > 0
  const long long t0 = clock64();
#endif
  for (;;) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
    if (done) return;
#if MK_MBAR_TIMEOUT_CYCLES > 0
    if (clock64() - t0 > MK_MBAR_TIMEOUT_CYCLES) __trap();
#endif
  }
}

__device__ __forceinline__ void tma_load_3d(const void* tmap, uint64_t* bar, void* dst, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          smem_u32(dst)),
      "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {  // arrives on `bar` when every MMA issued so far is done
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}

// shared-memory matrix descriptor (tcgen05): start >> 4 | LBO >> 4 << 16 | SBO >> 4 << 32 | version 1 << 46 | layout << 61
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
  return (uint64_t)((addr & 0x3FFFF) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
constexpr uint32_t LAYOUT_SW128_BASE32B = 1, LAYOUT_SW64 = 4;

// instruction descriptor, kind::tf32: D fp32, A tf32 K-major, B tf32 MN-major, M = 128, N = n
__device__ __forceinline__ uint32_t instr_desc(uint32_t n) {
  return (1u << 4) /*D = f32*/ | (2u << 7) /*A = tf32*/ | (2u << 10) /*B = tf32*/ | (0u << 15) /*A K-major*/ |
         (1u << 16) /*B MN-major*/ | ((n >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

struct TcParams {
  int n, nb, ld;        // receivers, bins, padded shots
  int ncols;            // 2 * ldf: valid real columns of S^
  int mt, ntl;          // tiles along M and N
  int nblk, stages;     // column blocks per B' tile, stages of the ring
  int mp;               // M tiles per CTA tile (1, or 2 when ncols <= 128: accumulator m lives in columns 128 m .. of the buffer)
  size_t s_row;         // floats between consecutive receivers of S^: nb * 2 ldf
  int dbg;              // TEMP experiment flags: 1 no TMA, 2 no split, 4 no MMA
};

__global__ void __launch_bounds__(kThreads, 1)
k_syn_gemm_tf32x3(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmBhi,
                  const __grid_constant__ CUtensorMap tmBlo, float* __restrict__ Shat, TcParams P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int STAGES = P.stages;
  const int MP = P.mp;
  const uint32_t STAGE_BYTES = stage_bytes(P.nblk, MP), B_BYTES = (uint32_t)P.nblk * BLK_BYTES, AREG = (uint32_t)MP * A_BYTES;
  const uint32_t TX_BYTES = AREG + 2 * B_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)STAGES * STAGE_BYTES);
  uint64_t* full = bars;                      // [kMaxStages] TMA landed
  uint64_t* empty = bars + kMaxStages;        // [kMaxStages] MMAs of the stage retired
  uint64_t* split = bars + 2 * kMaxStages;    // [kMaxStages] Alo written
  uint64_t* acc_full = bars + 3 * kMaxStages; // [2] chunk accumulator complete
  uint64_t* acc_empty = acc_full + 2;      // [2] chunk accumulator drained
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int per_bin = P.mt * P.ntl, ntiles = P.nb * per_bin;
  const int KB = (2 * P.ld) / BK;  // k'-blocks per tile

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, 1);
      mbar_init(split + s, 1);
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(acc_full + b, 1);
      mbar_init(acc_empty + b, kEpiWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {  // TMEM: all 512 columns (one CTA per SM)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------ TMA producer
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;  // ring position and its phase, kept incrementally (the ring length is a run-time value)
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int kk = t / per_bin, rem = t - kk * per_bin, mi = rem / P.ntl, ni = rem - mi * P.ntl;
        for (int kb = 0; kb < KB; ++kb) {
          mbar_wait(empty + s, ph ^ 1);
          uint8_t* st = smem + (size_t)s * STAGE_BYTES;
          if (P.dbg & 1) { mbar_arrive(full + s); if (++s == STAGES) { s = 0; ph ^= 1; } continue; }
          mbar_expect_tx(full + s, TX_BYTES);
          for (int m = 0; m < MP; ++m)  // rows past the last receiver arrive as zeros (and still count their bytes)
            tma_load_3d(&tmA, full + s, st + m * A_BYTES, kb * BK, kk, (mi * MP + m) * BM);
          tma_load_3d(&tmBhi, full + s, st + 2 * AREG, 0, kk * 2 * P.ld + kb * BK, ni * (BN / 32));
          tma_load_3d(&tmBlo, full + s, st + 2 * AREG + B_BYTES, 0, kk * 2 * P.ld + kb * BK, ni * (BN / 32));
          if (++s == STAGES) {
            s = 0;
            ph ^= 1;
          }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      uint32_t chunk_it = 0, ph = 0;
      int s = 0;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int rem = t % per_bin, ni = rem % P.ntl;
        int nmma = P.ncols - ni * BN;
        nmma = nmma > BN ? BN : ((nmma + 15) / 16) * 16;
        const uint32_t idesc = instr_desc((uint32_t)nmma);
        for (int kb0 = 0; kb0 < KB; kb0 += kChunkKb, ++chunk_it) {
          const int b = chunk_it & 1;
          mbar_wait(acc_empty + b, ((chunk_it >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint32_t d = tmem_base + (uint32_t)b * BN;
          const int kb1 = min(kb0 + kChunkKb, KB);
          for (int kb = kb0; kb < kb1; ++kb) {
            mbar_wait(full + s, ph);
            mbar_wait(split + s, ph);
            tc_fence_after();
            const uint32_t a_raw = smem_u32(smem + (size_t)s * STAGE_BYTES), a_lo = a_raw + AREG;
            const uint32_t b_hi = a_raw + 2 * AREG, b_lo = b_hi + B_BYTES;
#pragma unroll
            for (int j = 0; j < BK / UK; ++j) {
              if (P.dbg & 4) break;
              // A: K-major, 64-byte rows, SWIZZLE_64B: 8-row groups 512 B apart; a k'-chunk is 32 B further along the row
              const uint64_t da_raw = smem_desc(a_raw + j * 32, 16, 512, LAYOUT_SW64);
              const uint64_t da_lo = smem_desc(a_lo + j * 32, 16, 512, LAYOUT_SW64);
              const uint64_t da_raw1 = smem_desc(a_raw + A_BYTES + j * 32, 16, 512, LAYOUT_SW64);  // second M tile (MP = 2)
              const uint64_t da_lo1 = smem_desc(a_lo + A_BYTES + j * 32, 16, 512, LAYOUT_SW64);
              // B: MN-major tf32 must use the 128-byte swizzle with 32-byte atoms (the only MN-major layout the tensor
              //    core takes for 32-bit operands): [8 blocks of 32 columns][16 k' rows][128 B]; LBO = 2048 (next column
              //    block), SBO = 512 (next group of 4 k' rows); a k'-chunk of 8 rows is 1024 B further
              const uint64_t db_hi = smem_desc(b_hi + j * 1024, 2048, 512, LAYOUT_SW128_BASE32B);
              const uint64_t db_lo = smem_desc(b_lo + j * 1024, 2048, 512, LAYOUT_SW128_BASE32B);
              umma_tf32(d, da_lo, db_hi, idesc, (kb != kb0) || (j != 0));  // small terms first; a chunk starts from zero
              umma_tf32(d, da_raw, db_lo, idesc, 1);
              umma_tf32(d, da_raw, db_hi, idesc, 1);
              if (MP == 2) {
                umma_tf32(d + BN / 2, da_lo1, db_hi, idesc, (kb != kb0) || (j != 0));
                umma_tf32(d + BN / 2, da_raw1, db_lo, idesc, 1);
                umma_tf32(d + BN / 2, da_raw1, db_hi, idesc, 1);
              }
            }
            umma_commit(empty + s);
            if (++s == STAGES) {
              s = 0;
              ph ^= 1;
            }
          }
          umma_commit(acc_full + b);
        }
      }
    }
  } else if (warp < 4) {
    // ------------------------------------------------------------------------------------ split warps: Alo = A - tf32_trunc(A)
    // The two warps take ALTERNATE stages (a whole A tile each): the generic -> async proxy fence that must follow the
    // stores costs several hundred cycles, and this way two of them are in flight.
    const int sw = warp - 2;  // 0, 1
    int s = 0;
    uint32_t ph = 0, cnt = 0;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
      for (int kb = 0; kb < KB; ++kb, ++cnt) {
        if ((int)(cnt & 1) == sw) {
          mbar_wait(full + s, ph);
          if (P.dbg & 2) { if (lane == 0) mbar_arrive(split + s); if (++s == STAGES) { s = 0; ph ^= 1; } continue; }
          const float4* src = reinterpret_cast<const float4*>(smem + (size_t)s * STAGE_BYTES);
          float4* dst = reinterpret_cast<float4*>(smem + (size_t)s * STAGE_BYTES + AREG);
          constexpr int kPer = (int)(A_BYTES / 16) / 32;  // 16 float4 per lane and M tile
          for (int h = 0; h < 2 * MP; ++h) {
            float4 v[kPer / 2];
#pragma unroll
            for (int i = 0; i < kPer / 2; ++i) v[i] = src[lane + (h * (kPer / 2) + i) * 32];
#pragma unroll
            for (int i = 0; i < kPer / 2; ++i) {
              float4 l;
              l.x = v[i].x - __uint_as_float(__float_as_uint(v[i].x) & 0xffffe000u);
              l.y = v[i].y - __uint_as_float(__float_as_uint(v[i].y) & 0xffffe000u);
              l.z = v[i].z - __uint_as_float(__float_as_uint(v[i].z) & 0xffffe000u);
              l.w = v[i].w - __uint_as_float(__float_as_uint(v[i].w) & 0xffffe000u);
              dst[lane + (h * (kPer / 2) + i) * 32] = l;
            }
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the tensor core
          __syncwarp();
          if (lane == 0) mbar_arrive(split + s);
        }
        if (++s == STAGES) {
          s = 0;
          ph ^= 1;
        }
      }
    }
  } else {
    // ------------------------------------------------------------------------------------ epilogue: chunk sums in registers
    const int quad = warp & 3;        // TMEM lanes 32 quad .. 32 quad + 31 are the ones this warp may read
    const int half = (warp - 4) >> 2; // columns 128 half .. 128 half + 127 of the tile
    uint32_t chunk_it = 0;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
      const int kk = t / per_bin, rem = t - kk * per_bin, mi = rem / P.ntl, ni = rem - mi * P.ntl;
      // MP = 1: this warp's half of the 256 columns; MP = 2: the whole (<= 128-column) tile of M tile `half`
      const int cols = MP == 2 ? P.ncols : P.ncols - ni * BN - half * (BN / 2);  // valid columns (may exceed BN / 2, may be <= 0)
      float sum[BN / 2];
#pragma unroll
      for (int i = 0; i < BN / 2; ++i) sum[i] = 0.f;
      for (int kb0 = 0; kb0 < KB; kb0 += kChunkKb, ++chunk_it) {
        const int b = chunk_it & 1;
        mbar_wait(acc_full + b, (chunk_it >> 1) & 1);
        tc_fence_after();
        const uint32_t ta = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(b * BN + half * (BN / 2));
#pragma unroll
        for (int c = 0; c < BN / 32; ++c) {
          if (c * 16 < cols) {  // warp-uniform; columns past the MMA's N hold stale data
            uint32_t v[16];
            tmem_ld16(ta + (uint32_t)(c * 16), v);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int q = 0; q < 16; ++q) sum[c * 16 + q] += __uint_as_float(v[q]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(acc_empty + b);
      }
      const int r = (MP == 2 ? mi * 2 + half : mi) * BM + quad * 32 + lane;
      if (r < P.n) {
        float* dst = Shat + (size_t)r * P.s_row + (size_t)kk * P.ncols + (MP == 2 ? 0 : ni * BN + half * (BN / 2));
#pragma unroll
        for (int q = 0; q < BN / 8; ++q)
          if (q * 4 < cols)
            *reinterpret_cast<float4*>(dst + q * 4) = make_float4(sum[4 * q], sum[4 * q + 1], sum[4 * q + 2], sum[4 * q + 3]);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
}

// ---------------------------------------------------------------------------------------------- host: TMA descriptors
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode(mk_ctx* c, EncodeTiledFn* fn) {
  if (!c->encode_fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (int rc = check_cuda(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q), "cudaGetDriverEntryPoint"))
      return rc;
    if (q != cudaDriverEntryPointSuccess || !p) return set_err(c, MK_ERR_CUDA, "cuTensorMapEncodeTiled is not available");
    c->encode_fn = p;
  }
  *fn = reinterpret_cast<EncodeTiledFn>(c->encode_fn);
  return MK_OK;
}

int encode3(mk_ctx* c, EncodeTiledFn enc, void* out, const void* base, const cuuint64_t dims[3], const cuuint64_t strides[2],
            const cuuint32_t box[3], CUtensorMapSwizzle sw, const char* what) {
  const cuuint32_t es[3] = {1, 1, 1};
  const CUresult r = enc(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(base), dims,
                         strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[128];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", what, (int)r);
    return set_err(c, MK_ERR_CUDA, buf);
  }
  return MK_OK;
}

}  // namespace

bool tc_supported(const mk_ctx* c) {
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return false;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  return major == 10 && c->smem_optin >= 2 * stage_bytes(1, 1) + kSmemExtra;
}

int launch_syn_tc(mk_ctx* c, int slot, const float* d_Bhi, const float* d_Blo, float2* d_Shat, int nfoc, int ldf, int ldb) {
  (void)nfoc;
  EncodeTiledFn enc = nullptr;
  if (int rc = get_encode(c, &enc)) return rc;
  if (!c->tmap_A_ok) {
    // A' = R^ as fp32 [n][nb][2 ld]: dims (k', bin, r); box = 16 floats x 1 bin x 128 receivers; rows r >= n read as zero
    const cuuint64_t dims[3] = {(cuuint64_t)2 * c->ld, (cuuint64_t)c->nb, (cuuint64_t)c->nrow};  // local rows of R^
    const cuuint64_t str[2] = {(cuuint64_t)2 * c->ld * 4, (cuuint64_t)c->nb * 2 * c->ld * 4};
    const cuuint32_t box[3] = {BK, 1, BM};
    if (int rc = encode3(c, enc, c->tmap_A, c->d_Rhat, dims, str, box, CU_TENSOR_MAP_SWIZZLE_64B, "A")) return rc;
    c->tmap_A_ok = true;
  }
  const int nblk = std::min(BN / 32, (2 * ldf + 31) / 32);
  if (c->tmap_B_key[slot] != d_Bhi || c->tmap_B_ldb[slot] != ldb) {
    // B' plane [nb * 2 ld rows][ldb] seen as (column in block, row, column block): box = 32 x 16 x 8 lands in shared
    // memory as [8 column blocks][16 rows][128 B], the MN-major SWIZZLE_128B_BASE32B operand layout
    const cuuint64_t dims[3] = {32, (cuuint64_t)c->nb * 2 * c->ld, (cuuint64_t)ldb / 32};
    const cuuint64_t str[2] = {(cuuint64_t)ldb * 4, 128};
    const cuuint32_t box[3] = {32, BK, (cuuint32_t)nblk};  // ldb is a function of nfoc, so is nblk: one cache key
    if (int rc = encode3(c, enc, c->tmap_B[slot][0], d_Bhi, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, "B hi")) return rc;
    if (int rc = encode3(c, enc, c->tmap_B[slot][1], d_Blo, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, "B lo")) return rc;
    c->tmap_B_key[slot] = d_Bhi;
    c->tmap_B_ldb[slot] = ldb;
  }
  TcParams P;
  { const char* e = getenv("MK_TC_DEBUG"); P.dbg = e ? atoi(e) : 0; }
  P.n = c->nrow;  // row sharding: local rows; S^ is offset to the first one below
  P.nb = c->nb;
  P.ld = c->ld;
  P.ncols = 2 * ldf;
  const int mtiles = (c->nrow + BM - 1) / BM;
  P.mp = (2 * ldf <= BN / 2 && mtiles >= 2) ? 2 : 1;
  P.mt = (mtiles + P.mp - 1) / P.mp;
  P.ntl = (P.ncols + BN - 1) / BN;
  P.s_row = (size_t)c->nb * 2 * ldf;
  P.nblk = nblk;
  P.stages = (int)std::min<size_t>(kMaxStages, (c->smem_optin - kSmemExtra) / stage_bytes(nblk, P.mp));
  if (P.stages < 2) return set_err(c, MK_ERR_INVALID_ARG, "not enough shared memory for the tcgen05 contraction");
  const size_t kSmemBytes = (size_t)P.stages * stage_bytes(nblk, P.mp) + kSmemExtra;
  if (int rc = check_cuda(c, cudaFuncSetAttribute(k_syn_gemm_tf32x3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes),
                          "cudaFuncSetAttribute"))
    return rc;
  const int ntiles = P.nb * P.mt * P.ntl;
  const int grid = ntiles < c->num_sms ? ntiles : c->num_sms;
  k_syn_gemm_tf32x3<<<grid, kThreads, kSmemBytes, c->stream>>>(*reinterpret_cast<const CUtensorMap*>(c->tmap_A),
                                                               *reinterpret_cast<const CUtensorMap*>(c->tmap_B[slot][0]),
                                                               *reinterpret_cast<const CUtensorMap*>(c->tmap_B[slot][1]),
                                                               reinterpret_cast<float*>(d_Shat + (size_t)c->r0 * c->nb * ldf), P);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_syn_gemm_tf32x3");
}

}  // namespace mk
