// mk_syn_tc.cu — synthesis contraction for large focal batches on the 5th-generation tensor cores (SURVEY.md §8(f)
// NEXT-2; BASELINE.json north_star (b): "a tcgen05/TMEM 3xTF32 split path only if it meets the FP32 tolerance").
//
// Per bin k the complex GEMM  S^_k[r][f] = sum_s R^_k[r][s] N^_k[s][f]  (eq. (1)) is run as the REAL GEMM
//     C'[r][2f+c] = sum_s ( Re R^[r][s] * B0[s][2f+c] + Im R^[r][s] * B1[s][2f+c] ),     c = (0: re, 1: im)
//   B0[s] = the row N^[k][s][.] read as interleaved floats (re, im)  — the operand exactly as the transform kernels
//           store it for every regime, [nb][ld][ldf] complex64 (TMA, no copy, no second plane in HBM);
//   B1[s] = i N^[k][s][.] = (-im, re): the same row rotated by 90 degrees, made in shared memory;
//   A     = the row R^[r][k][.] exactly as it sits in HBM (K-major, TMA lands it in shared memory); the split warps
//           read it ONCE, de-interleave its (re, im) pairs four shots at a time in registers and store it into TENSOR
//           MEMORY (tcgen05.st): the MMAs take A from TMEM, so that one K = 8 step reads (re s..s+3 | im s..s+3) of A
//           against (B0 rows s..s+3 | B1 rows s..s+3) of B;
//   C'    = S^[r][k][.] as interleaved floats — the layout k_post reads.
// 3xTF32: x = hi + lo with hi = the tf32 the tensor core sees when it reads the fp32 word (the low 13 mantissa bits are
// not used) and lo = x - hi (exact in fp32, then rounded to nearest tf32); every K step issues  A_lo*B_hi + A_hi*B_lo + A_hi*B_hi  into one fp32
// accumulator in TMEM.  The dropped term A_lo*B_lo is O(2^-21) relative.  Only raw fp32 words cross HBM and L2: the lo
// parts, the rotation and the de-interleave are computed per stage by the split warps from the tile TMA delivered.
//
// Accumulation.  The tensor core adds into its fp32 accumulator with TRUNCATION, not round-to-nearest: measured on B200
// with one accumulator over the whole K extent the relative error of S^ grows linearly with the number of MMA steps
// (about 2e-8 per step: 6.8e-7 at n = 32, 2.9e-5 at n = 2048, against 1.2e-6 for the FFMA kernel), which breaks the
// 2e-5 per-iteration tolerance from n ~ 600 on.  So K is cut into CHUNKS of kChunk stages (24 MMA steps): every chunk
// starts a fresh TMEM accumulator, and the read-out warps add the finished chunk into fp32 registers (round-to-nearest)
// while the tensor core works on the next chunk in the other TMEM buffer.  The error is then that of one chunk
// (~5e-7), independent of n.
//
// What shaped it (measured on B200, round 2, config 2 = 601 x 608 x 451 bins x 601 focal points; the
// MK_OPT_TUNE switches that leave out one part of the kernel at a time are still in the code):
//   * tcgen05.mma kind::tf32 M = 128, K = 8 takes N / 2 clk per instruction with nothing else going on;
//   * an mbarrier wait in the ISSUING thread is not free: the thread runs only ~4 MMAs ahead of the pipe and a try_wait
//     costs 70-90 clk that the pipe then idles.  The issuing thread therefore never touches an mbarrier: readiness
//     reaches it through plain shared-memory counters (release / acquire) that it polls between bursts of MMAs;
//   * THE FEED, not the math, paced every earlier version (~1100-1400 clk per 8-shot stage whatever N, ring depth or split
//     arrangement; with MMAs, split and read-out all switched off the kernel still took 4.3 of 5.1 ms).  The TMA unit
//     charges per ROW of a box, about 8 clk whether the row has 64 or 128 bytes: the A tile of one stage (128 receivers x
//     64 bytes) alone cost 1030 clk, more than the stage's six MMAs (576).  Hence
//       - A boxes of 16 shots (128-byte rows, the swizzle span) in a ring of their own, one box per two stages;
//       - B delivered as 8 dense rows of <= 768 bytes per stage instead of 8 nblk rows in the tensor core's layout; the
//         split warps, who read every element anyway, write the MN-major swizzled planes themselves;
//     A-only feed 4.25 -> 2.72 ms;
//   * the raw rings (A: 3 .. 12 boxes of two stages each, as many as shared memory allows; B: <= 8 tiles) run ahead of the
//     four operand stages by their own length, so the latency of the loads is not inside the loop the MMAs close
//     (empty -> split -> ready -> MMA -> empty);
//   * with R^ in its TILED layout (MK_OPT_RHAT_LAYOUT = 1: the box is 16 KB contiguous in HBM, stored pre-swizzled) the
//     producer issues one cp.async.bulk per box instead of a TMA box of 128 rows that lie 2 MB apart: config 2 4.23 -> 4.12 ms
//     per contraction, DRAM traffic 6.1 -> 4.3 GB (3.9 algorithmic), config 4 146 -> 105 GB;
//   * A IN TENSOR MEMORY: with both operands in shared memory the MMAs read 6 x (4 KB of A + 8 KB of B) per stage and the
//     split warps moved 56 KB more; now the MMAs read only B, the split warps read A once and tcgen05.st it, and A_hi /
//     A_lo occupy no shared memory (which is what pays for the raw rings);
//   * one stage's split is a LATENCY chain (waits, LDS -> ALU -> STS / tcgen05.st, tcgen05.wait::st, proxy fence, arrive:
//     ~1400 clk for ~250 instructions per warp), so three groups of four warps take the stages in rotation;
//   * a waiting warp must really sleep: with the default suspend time the read-out warps' try_wait loops were 40 % of all
//     instructions issued on the SM (same schedulers as the split warps); try_wait now carries a suspend-time hint;
//   * NOT the depth of the operand ring: with every load, MMA, split and read-out switched off the barrier chain alone
//     (empty[s] -> split -> split_bar -> relay -> ready -> MMA issue -> tcgen05.commit) takes 1.83 ms = 443 clk per stage,
//     but N tiles of 128 columns with EIGHT operand stages (-DMK_TC_BN=128) are slower on every config (config 2 4.94 ms,
//     config 3 5.33, config 4 70.1 against 4.21 / 5.20 / 66.7), and waking the waiters without a suspend hint changes
//     nothing.  What holds config 3 at ~650 clk per stage against 384 clk of MMAs is not identified;
//   * the chip is POWER-bound under this kernel (1000 W cap: 1.6-1.8 GHz): every byte through L2, every byte through shared
//     memory and every spinning warp costs SM clock.
// Result: tensor pipe 55 % -> 68-69 % active (config 4: 78-81 %), config 2 4.74 -> 4.12 ms, config 3 7.35 -> 5.28 ms per contraction.
//
// Tensor memory (512 columns): two chunk accumulators of BN = 192 columns, and a ring of four A slots of 32 columns
// (per K step 8 columns of A_hi and 8 of A_lo; lane = receiver row of the tile).
//
// Kernel: persistent, one CTA per SM, warp-specialised, 768 threads = 6 warpgroups with their own register budgets
// (setmaxnreg: the kernel starts at 80 registers per thread; control 32, split 64, read-out 128) —
//   warp 0      producer of the raw A boxes [128 receivers][16 shots]: TMA (SWIZZLE_128B) from the row-major R^, one bulk copy from
//               the tiled R^; ring of 3 .. 12
//   warp 3      TMA producer of the raw B tiles [8 shots][<= 192 floats] (dense rows), ring of <= 8
//   warp 1      tcgen05.mma issuer (one thread): kind::tf32, M = 128, N <= 192, K = 8, A from TMEM, B from shared memory;
//               tcgen05.commit releases the operand stage / publishes the chunk
//   warp 2      relay: split_bar[stage] (mbarrier) -> ready[stage] (the word the MMA warp polls)
//   warps 4-15  split warps, three groups of four; group g takes the stages g, g + 3, ...  A: thread = row of the tile: four
//               128-bit loads of its half of the box, lo parts, two tcgen05.st of 16 columns.  B: raw tile -> B0_hi, B0_lo,
//               B1_hi, B1_lo in the tensor core's layout.  tcgen05.wait::st, proxy fence, arrive on split_bar[stage] and
//               on the raw rings' empty barriers
//   warps 16-23 read-out warps.  Per chunk: tcgen05.ld of the finished accumulator (warp w owns TMEM lanes 32 (w % 4) .. +31
//               and the column half (w - 16) / 4) -> += 96 running sums in registers, drained += 1 per warp; per tile:
//               128-bit global stores of S^
#include <cuda.h>

#include <algorithm>

#include "mk_internal.cuh"

namespace mk {

namespace {

// MK_TC_K16 = 1: a stage is 16 shots (one whole A box, two 8-shot sub-stages of B planes, 12 MMAs) and the N tile 128 columns
// (tensor memory: 2 x 128 accumulator columns + 4 x 64 columns of A); 0: 8-shot stages, N tile MK_TC_BN.  Measured: half as
// many, fatter stages change nothing (config 2 4.46 ms, config 3 5.18, config 4 67.1, narrow batches 367 us against 4.02 /
// 5.21 / 64.0 / 354): the cost is not per stage.
#ifndef MK_TC_K16
#define MK_TC_K16 0
#endif
#ifndef MK_TC_BN
#define MK_TC_BN (MK_TC_K16 ? 128 : 192)
#endif
constexpr int BM = 128;         // rows (receivers) per tile = TMEM lanes
constexpr int BN = MK_TC_BN;    // real columns (2 per focal point) per tile = TMEM columns per accumulator (128 or 192)
constexpr int BKC = 8;          // shots (complex k) per stage
constexpr int kMaxRawB = 8;     // ring of raw B tiles: as many as fit (8 at N = 192)
constexpr int kSub = MK_TC_K16 ? 2 : 1;  // 8-shot sub-stages per stage
constexpr int kTmemSlots = (MK_TC_BN == 128 && !MK_TC_K16) ? 8 : 4, kLgSlots = (MK_TC_BN == 128 && !MK_TC_K16) ? 3 : 2;  // ring of operand stages: stage it uses A slot it % 4 in tensor memory and B planes it % 4 in shared
                                // memory, both free once the MMAs of stage it - 4 retired
constexpr int kSplitWarps = 4, kSplitThreads = 32 * kSplitWarps;  // per split group
#ifndef MK_TC_SPLIT_GROUPS
#define MK_TC_SPLIT_GROUPS 3
#endif
constexpr int kSplitGroups = MK_TC_SPLIT_GROUPS;  // group g takes the stages g, g + G, g + 2 G, ...
constexpr int kReadWarps = 8;
constexpr int kFirstReadWarp = 4 + kSplitGroups * kSplitWarps;
constexpr int kThreads = 128 + kSplitGroups * kSplitThreads + 32 * kReadWarps;  // 24 warps = 6 warpgroups: {TMA A, MMA, relay, TMA B}, split x 3, read-out x 2
// Register budget per warpgroup (setmaxnreg): launched at 80 registers per thread (768 x 80 = 61440 is the CTA's pool); the
// control warpgroup gives most of its share back and the read-out warps, who hold 96 running sums each, take it:
// 128 x 32 + 384 x 64 + 256 x 128 = 61440.  (Two split groups: 640 threads at 96; 128 x 32 + 256 x 72 + 256 x 152.)
// (Four split groups, -DMK_TC_SPLIT_GROUPS=4: 896 threads at 72 = 64512; 128 x 32 + 512 x 56 + 256 x 120 = 63488.  Measured: no
// gain - narrow batches 347 us against 340, config 2 4.25 ms per contraction against 4.12: three groups already keep up.)
constexpr int kRegsControl = 32, kRegsSplit = kSplitGroups == 3 ? 64 : (kSplitGroups == 4 ? 56 : 72),
              kRegsRead = kSplitGroups == 3 ? 128 : (kSplitGroups == 4 ? 120 : 152);
#ifndef MK_TC_READ16
#define MK_TC_READ16 1
#endif
#ifndef MK_TC_CHUNK
#define MK_TC_CHUNK (4 / kSub)
#endif
constexpr int kChunk = MK_TC_CHUNK;  // stages per accumulation chunk (24 MMA steps)
#ifndef MK_TC_A_LDG
#define MK_TC_A_LDG 0
#endif
// How the A tile reaches the split warps: 0 = TMA boxes of 16 shots into a shared-memory ring (the TMA unit's per-row cost
// makes this the slowest part of the feed, 128 rows per box ~ 1000-1300 clk, but it runs 3 boxes ahead); 1 = every split
// thread loads the 64 bytes of its receiver row straight from global memory (four 128-bit ld.global.nc issued before the
// stage's other waits; no TMA, no shared memory for A).  Measured: 1 is far slower (config 2 5.7 ms, config 3 21.3 ms,
// config 4 286 ms against 4.2 / 5.3 / 66): with one stage per split group in flight the ~1.5 us of a load from HBM sits in
// the chain of every stage; the register budget of the split warps has no room for the 4-6 stages of prefetch that TMA
// gives for free.
constexpr bool kALdg = MK_TC_A_LDG == 1;
// MK_TC_A_LDG = 2: the A ring is filled by cp.async (LDGSTS) of the whole producer warp instead of one TMA instruction:
// per box 32 instructions of 32 lanes x 16 bytes (8 lanes = one 128-byte row, 4 rows per instruction), written in the same
// swizzled layout, completion through cp.async.mbarrier.arrive on the box's full barrier.
constexpr bool kACpAsync = MK_TC_A_LDG == 2;
constexpr int kMinASlots = kALdg ? 0 : 3, kMaxASlots = kALdg ? 0 : 12;  // ring of raw A boxes: as many as fit (bytes in flight per SM are
                                                                          // what the rate of R^ from HBM follows: 3 boxes = 48 KB gave 3.5 TB/s)
constexpr uint32_t A_BOX_BYTES = BM * 4 * BKC * 4;  // 16 KB: one raw A box = [128 rows][16 shots] = two stages, 128-byte rows
constexpr uint32_t BLK_BYTES = BKC * 32 * 4;    // 1 KB: one 32-column block of one B region (8 rows of 128 B)
// Shared memory: the ring of raw A boxes; the ring of raw B tiles as TMA delivered them ([8 shots][nblk x 128 B], dense
// rows); four operand stages of four B regions of nblk column blocks each that the tensor core reads: B0_hi, B0_lo,
// B1_hi, B1_lo; nblk = min(6, columns / 32).  The distance B0 -> B1 (two regions) is the stride-byte-offset of the B
// descriptors: the second group of four K rows of every MMA is the rotated copy of the first.  The raw rings run ahead of
// the operand stages by their own length: the latency of the loads is not in the loop that the MMAs close.
__host__ __device__ constexpr uint32_t planes_bytes(int nblk) { return kSub * 4 * (uint32_t)nblk * BLK_BYTES; }
__host__ __device__ constexpr uint32_t fixed_smem(int nblk) { return kMinASlots * A_BOX_BYTES + kTmemSlots * planes_bytes(nblk); }
constexpr size_t kSmemExtra = 1024 /*alignment slack*/ + 512 /*barriers, counters: (2 x 8 + 2 x 8 + 2 + 2 x 12) x 8 + (8 + 2 + 1) x 4 bytes*/;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kTmemA = 2 * BN;  // first column of the A ring
constexpr uint32_t kTmemAStage = 32 * kSub; // columns per slot: K step j at 16 j: A_hi (8 columns), A_lo (8 columns)
static_assert(kTmemA + kTmemSlots * kTmemAStage <= kTmemCols, "tensor memory budget");

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
// Bounded waits: a protocol bug traps (the launch fails with an error) instead of hanging the GPU.  The budget is a
// compile-time option: MK_MBAR_TIMEOUT_CYCLES (default 4e10 SM cycles, about 20 s — no stage of a healthy launch waits
// that long, not even under a profiler's replay or on a contended GPU); -DMK_MBAR_TIMEOUT_CYCLES=0 compiles the
// check out.
#ifndef MK_MBAR_TIMEOUT_CYCLES
#define MK_MBAR_TIMEOUT_CYCLES 40000000000LL
#endif
// try_wait suspends the thread in hardware until the phase completes or a time limit passes.  The default limit is short:
// measured (ncu, round 2) the eight read-out warps came back every ~75 clk and their retry loops were 40 % of all the
// instructions the SM issued, taking issue slots from the split warps on the same schedulers.  With an explicit limit the
// thread sleeps until the barrier wakes it.
constexpr uint32_t kSuspendHintNs = 20000;
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
#if MK_MBAR_TIMEOUT_CYCLES > 0
  const long long t0 = clock64();
#endif
  for (;;) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity), "r"(kSuspendHintNs)
        : "memory");
    if (done) return;
#if MK_MBAR_TIMEOUT_CYCLES > 0
    if (clock64() - t0 > MK_MBAR_TIMEOUT_CYCLES) __trap();
#endif
  }
}
// MK_TC_PROBE = 1 (diagnosis only): every role of CTA 0 sums the clocks it spends in each of its waits and prints them.
// Round 2, config 2 (8106 stages on CTA 0, 835 clk per stage): the producers wait 73 %, the relay 85 %, the read-out
// warps 49 %, the MMA issuer 42 % (35 % for a stage to become ready, 7 % for a drained accumulator); the split groups wait
// 28 % (6 % + 6 % for raw tiles that are long there, 16 % for the operand stage to come free) and WORK the rest: ~1800 clk
// per stage and group (narrow batches: ~1040), i.e. 600 clk per stage over three groups against 576 clk of MMAs.  The
// split warps pace the kernel; a fourth group does not help (the groups share the schedulers and the shared-memory pipe,
// 61 % and 70 % busy in ncu), so the next step is less split work per stage, not more warps.
#ifndef MK_TC_PROBE
#define MK_TC_PROBE 0
#endif
#if MK_TC_PROBE
#define PROBE_DECL long long pw_[3] = {0, 0, 0}; const long long pt0_ = clock64()
#define PROBE_WAIT(i, ...) do { const long long a_ = clock64(); __VA_ARGS__; pw_[i] += clock64() - a_; } while (0)
#define PROBE_PRINT(name) do { if (blockIdx.x == 0) printf("%-12s total %9lld  wait0 %9lld  wait1 %9lld  wait2 %9lld\n", name, clock64() - pt0_, pw_[0], pw_[1], pw_[2]); } while (0)
#else
#define PROBE_DECL
#define PROBE_WAIT(i, ...) do { __VA_ARGS__; } while (0)
#define PROBE_PRINT(name)
#endif
// non-blocking look at a barrier's phase (the two raw-tile barriers of a stage are asked together, see the split warps)
__device__ __forceinline__ uint32_t mbar_test(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return done;
}
// (MK_TC_TEST2 = 1.  Measured: neutral - narrow batches 327.6 us against 327, 128 focal points 955 against 973, config 2
// 4.09 ms per contraction against 4.12, inside the run-to-run spread; off.)
#ifndef MK_TC_TEST2
#define MK_TC_TEST2 0
#endif
// A whole warp waiting on one barrier costs ~150 clk even when the phase is long complete (measured with MK_TC_PROBE: the
// three waits of a split group are ~450 of the ~2500 clk it spends per stage).  MK_TC_WARP_WAIT = 1 lets one lane wait and
// the others join it at a __syncwarp: SLOWER (CTA 0 of config 2: 7.60 M clk against 6.77 M; narrow batches 812 k against
// 680 k), the divergence costs more than the 31 redundant try_waits.  Off.
#ifndef MK_TC_WARP_WAIT
#define MK_TC_WARP_WAIT 0
#endif
__device__ __forceinline__ void mbar_wait_warp(uint64_t* bar, uint32_t parity) {
#if MK_TC_WARP_WAIT
  if ((threadIdx.x & 31) == 0) mbar_wait(bar, parity);
  __syncwarp();
#else
  mbar_wait(bar, parity);
#endif
}
// shared-memory counters that carry readiness to the MMA-issuing thread (see the header: no mbarrier there)
__device__ __forceinline__ void flag_add(uint32_t* p) {
  asm volatile("red.release.cta.shared::cta.add.u32 [%0], 1;" ::"r"(smem_u32(p)) : "memory");
}
__device__ __forceinline__ void flag_set(uint32_t* p, uint32_t v) {
  asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void flag_wait_ge(const uint32_t* p, uint32_t need) {
  const uint32_t addr = smem_u32(p);
#if MK_MBAR_TIMEOUT_CYCLES > 0
  long long t0 = 0;
#endif
  for (;;) {
    uint32_t v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    if ((int32_t)(v - need) >= 0) return;
#if MK_MBAR_TIMEOUT_CYCLES > 0
    if (t0 == 0) t0 = clock64();
    else if (clock64() - t0 > MK_MBAR_TIMEOUT_CYCLES) __trap();
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

__device__ __forceinline__ void tma_load_2d(const void* tmap, uint64_t* bar, void* dst, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(smem_u32(dst)),
               "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
               : "memory");
}

__device__ __forceinline__ void bulk_load(uint64_t* bar, void* dst, const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
               "r"(smem_u32(bar))
               : "memory");
}

__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }

// A from tensor memory, B from shared memory; the B descriptor given as 32-bit halves: the high word (SBO, version,
// layout) never changes and the low word (start address, LBO) of a stage is that of stage 0 plus a constant, so the
// issuing warp keeps them in (uniform) registers and pays one add per descriptor and stage
__device__ __forceinline__ void umma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint32_t b_lo32, uint32_t b_hi32, uint32_t idesc,
                                             uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 db;\n\t"
      "mov.b64 db, {%2, %3};\n\t"
      "setp.ne.b32 p, %5, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], db, %4, p;\n\t}" ::"r"(tmem_d),
      "r"(tmem_a), "r"(b_lo32), "r"(b_hi32), "r"(idesc), "r"(accumulate)
      : "memory");
}
// one lane of a fully active warp (the same one every time: tcgen05.commit tracks the MMAs of the thread that runs it)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {  // arrives on `bar` when every MMA issued so far is done
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float4& a, const float4& b, const float4& c, const float4& d) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
      "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w), "f"(c.x), "f"(c.y), "f"(c.z), "f"(c.w), "f"(d.x),
      "f"(d.y), "f"(d.z), "f"(d.w)
      : "memory");
}
// eight columns at a time: the read-out warps hold 96 running sums each
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t* v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}

// sixteen columns with one instruction (MK_TC_READ16 = 1, the default: the read-out of a chunk is a chain of load -> wait ->
// add round trips and the issuer waits for it two chunks later; half as many round trips: narrow batches 340 -> 327 us,
// 128 / 256 focal points on config 1's R^ 987 -> 973 / 1642 -> 1624 us; same sums in the same order)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
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

// explicit shared-space accesses with 32-bit addresses (after the alignment arithmetic on the dynamic shared-memory
// base the compiler no longer knows the space and would emit generic 64-bit loads and stores)
__device__ __forceinline__ float4 ldg128_stream(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, float4 v) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// lo = x - hi is exact in fp32 and can have 13 significant bits; the tensor core TRUNCATES it to the 11 of tf32 (it does not
// use the low 13 bits of the word), a bias of ~2^-23 |x| with the sign of x on every operand, i.e. a coherent relative
// shrink of every product that adds up over the Neumann iterations (measured: 8e-6 after 8 iterations against 1e-6 for
// the FFMA kernel).  Adding half a tf32 ulp to the magnitude here (one integer add on the sign-magnitude word) turns the
// tensor core's truncation into round-to-nearest and the remaining error is unbiased.  Three instructions per element:
// the split warps' instruction stream is what paces the kernel (ncu, round 2: they were busy 94 % of the time).
__device__ __forceinline__ float lo_part(float x) {
  const float l = x - __uint_as_float(__float_as_uint(x) & 0xffffe000u);
  return __uint_as_float(__float_as_uint(l) + 0x1000u);
}
__device__ __forceinline__ float4 lo4(float4 v) { return make_float4(lo_part(v.x), lo_part(v.y), lo_part(v.z), lo_part(v.w)); }

struct TcParams {
  int n, nb, ld;        // receivers (rows of R^ this context owns), bins, padded shots
  int ncols;            // 2 * ldf: real columns of S^ (a multiple of 32)
  int mt, ntl;          // tiles along M and N; N tile ni covers the 32-column blocks [ni nblocks / ntl, (ni + 1) nblocks / ntl):
                        // widths differ by at most one block, so the CTAs that share an A tile run in step and meet in L2
  int nblocks;          // ncols / 32
  int nblk, nrb, na;    // column blocks per B region, slots of the raw B ring, slots of the raw A ring
  size_t s_row;         // floats between consecutive receivers of S^: nb * 2 ldf
  const float4* Rhat4;  // kALdg: the row block of R^ as float4; receiver row r, bin kk, shots 8 kb .. 8 kb + 7 = 4 float4 at
  size_t a_row4;        //   Rhat4 + r a_row4 + kk ld4 + 4 kb   (a_row4 = nb ld / 2, ld4 = ld / 2)
  int ld4;
  int a_tiled;          // R^ is stored in 16 KB boxes (MK_OPT_RHAT_LAYOUT = 1): one bulk copy per box
  uint32_t* progress;   // [grid] raw A boxes each CTA has asked for (zeroed before the launch); NULL when ntl == 1
  int tune;             // MK_OPT_TUNE bits 2..5: parts of the kernel left out (bottleneck measurements; results are wrong)
};

__device__ __forceinline__ int tile_col0(const TcParams& P, int ni) { return 32 * ((ni * P.nblocks) / P.ntl); }

__global__ void __launch_bounds__(kThreads, 1)
k_syn_gemm_tf32x3(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, float* __restrict__ Shat,
                  TcParams P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int NRB = P.nrb;
  const uint32_t REG = (uint32_t)P.nblk * BLK_BYTES, SUBPL = 4 * REG, PLANES = kSub * SUBPL, RAW = kSub * REG;  // REG: bytes of one B region of 8 shots
  const int kASlots = P.na;
  uint8_t* planes = smem + (size_t)kASlots * A_BOX_BYTES;            // the A ring comes first, then the operand stages,
  uint8_t* rawB = planes + (size_t)kTmemSlots * PLANES;      // then the raw B ring
  uint64_t* bars = reinterpret_cast<uint64_t*>(rawB + (size_t)NRB * RAW);
  uint64_t* fullB = bars;                          // [kMaxRawB] raw B tile landed
  uint64_t* emptyB = bars + kMaxRawB;              // [kMaxRawB] the split group that took the stage has read it
  uint64_t* empty = bars + 2 * kMaxRawB;           // [kTmemSlots] MMAs of the operand stage retired
  uint64_t* split_bar = empty + kTmemSlots;        // [kTmemSlots] the split warps are done with the stage
  uint64_t* acc_full = split_bar + kTmemSlots;     // [2] chunk accumulator complete
  uint64_t* fullA = acc_full + 2;                  // [kASlots] raw A box landed
  uint64_t* emptyA = fullA + kMaxASlots;           // [kASlots] both halves of the box have been read
  uint32_t* ready = reinterpret_cast<uint32_t*>(emptyA + kMaxASlots);  // [kTmemSlots] uses of the stage that are ready for the MMAs (relay)
  uint32_t* drained = ready + kTmemSlots;      // [2] read-out warps done with a use of TMEM buffer b (counts up; PER BUFFER:
                                               // one sum over both would let fast warps' arrivals for the other buffer stand in for
                                               // a slow warp's missing one)
  uint32_t* tmem_slot = drained + 2;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // warp-uniform by construction
  const int per_bin = P.mt * P.ntl, ntiles = P.nb * per_bin;
  const int KB = P.ld / (BKC * kSub);  // stages per tile

  if (threadIdx.x == 0) {
    for (int s = 0; s < NRB; ++s) {
      mbar_init(fullB + s, 1);  // the B producer
      mbar_init(emptyB + s, kSplitWarps);
    }
    for (int s = 0; s < kTmemSlots; ++s) {
      mbar_init(empty + s, 1);
      mbar_init(split_bar + s, kSplitWarps);
      ready[s] = 0;
    }
    mbar_init(acc_full + 0, 1);
    mbar_init(acc_full + 1, 1);
    for (int a = 0; a < kASlots; ++a) {
      mbar_init(fullA + a, kACpAsync ? 32 : 1);
      mbar_init(emptyA + a, (2 / kSub) * kSplitWarps);  // 8-shot stages: the box has two halves = two stages, each read by the four warps of one group
    }
    drained[0] = drained[1] = 0;
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

  // (each role's branch opens with its own setmaxnreg: ptxas budgets a branch by the setmaxnreg that dominates it)
  if (warp == 0) {
    // ------------------------------------------------------------------------------------ TMA producer
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
    // One box = [128 receivers][16 shots] = 128 rows of 128 bytes (SWIZZLE_128B) feeds two stages: the TMA unit's cost is
    // per ROW of a box (measured: ~8 clk per row whether it has 64 or 128 bytes; 128 rows x 64 B per 8-shot stage alone
    // took 1030 clk, more than the stage's MMAs), so rows are made as long as the swizzle span allows.
    // The ntl CTAs that work on the N tiles of one (bin, receiver tile) read the SAME A boxes.  Left alone they drift apart
    // by more than the L2 holds (measured on config 4: 155 GB from DRAM per launch for 62 GB of operands: every N tile
    // reads R^ from HBM again).  MK_OPT_TUNE bit 10 keeps them in step — the grid is a multiple of ntl, CTA b's siblings
    // are the ntl-aligned group around it (same tiles, other ni), every CTA publishes how many boxes it has asked for and
    // nobody runs more than kLead boxes ahead of its slowest sibling — and DRAM reads do drop (155 -> 104 GB), but every
    // CTA then moves at the pace of the momentarily slowest of its group: config 4 66 -> 82 ms, config 2 4.2 -> 5.3 ms.
    // Off by default; the remedy that does not couple the CTAs' pace is a cluster with the A box multicast (not built).
    if (kACpAsync) {
      int a = 0;
      uint32_t ph = 0;
      const int KB2 = KB * kSub / 2;  // A boxes per tile
      const int sub = lane >> 3, ch = lane & 7;  // this lane: rows sub, sub + 4, ..., 16-byte chunk ch of the 128-byte row
      const uint32_t a_smem = smem_u32(smem);
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int kk = t / per_bin, rem = t - kk * per_bin, mi = rem / P.ntl;
        for (int kb2 = 0; kb2 < KB2; ++kb2) {
          mbar_wait(emptyA + a, ph ^ 1);
          const uint32_t dst0 = a_smem + (uint32_t)a * A_BOX_BYTES;
#pragma unroll 8
          for (int i = 0; i < BM / 4; ++i) {
            const int row = 4 * i + sub, r = mi * BM + row;
            const bool in = r < P.n;
            const float4* src = P.Rhat4 + (size_t)(in ? r : 0) * P.a_row4 + (size_t)kk * P.ld4 + 8 * kb2 + ch;
            const uint32_t dst = dst0 + (uint32_t)row * 128 + (uint32_t)((ch ^ (row & 7)) << 4);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(in ? 16 : 0) : "memory");  // rows past the last receiver: zeros
          }
          asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(fullA + a)) : "memory");
          if (++a >= kASlots) {
            a = 0;
            ph ^= 1;
          }
        }
      }
    } else if (lane == 0 && !kALdg) {
      int a = 0;
      uint32_t ph = 0;  // ring position and its phase
      const int KB2 = KB * kSub / 2;  // A boxes per tile
      uint32_t q = 0;   // boxes asked for so far
      PROBE_DECL;
      const int sib0 = (int)blockIdx.x - (int)blockIdx.x % P.ntl;
      constexpr uint32_t kLead = 16, kEvery = 8;  // looked at every 8th box only: a look is ntl - 1 round trips to L2
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int kk = t / per_bin, rem = t - kk * per_bin, mi = rem / P.ntl;
        for (int kb2 = 0; kb2 < KB2; ++kb2, ++q) {
          if (P.progress && q >= kLead && q % kEvery == 0) {
#if MK_MBAR_TIMEOUT_CYCLES > 0
            const long long t0 = clock64();
#endif
            for (int j = 0; j < P.ntl; ++j) {
              if (sib0 + j == (int)blockIdx.x) continue;
              for (;;) {
                uint32_t v;
                asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(P.progress + sib0 + j) : "memory");
                if (v + kLead > q) break;
#if MK_MBAR_TIMEOUT_CYCLES > 0
                if (clock64() - t0 > MK_MBAR_TIMEOUT_CYCLES) __trap();
#endif
              }
            }
          }
          PROBE_WAIT(0, mbar_wait(emptyA + a, ph ^ 1));
          if (P.tune & (64 | 128)) {
            mbar_arrive(fullA + a);
          } else {
            mbar_expect_tx(fullA + a, A_BOX_BYTES);
            if (P.a_tiled)  // the box is 16 KB contiguous in HBM, already in the swizzled layout (rows past the last receiver are stored zeros)
              bulk_load(fullA + a, smem + (size_t)a * A_BOX_BYTES,
                        reinterpret_cast<const uint8_t*>(P.Rhat4) + (((size_t)mi * P.nb + kk) * KB2 + kb2) * A_BOX_BYTES, A_BOX_BYTES);
            else
              tma_load_3d(&tmA, fullA + a, smem + (size_t)a * A_BOX_BYTES, kb2 * 4 * BKC, kk, mi * BM);  // rows past the last receiver arrive as zeros
          }
          if (P.progress && (q + 1) % kEvery == 0)
            asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(P.progress + blockIdx.x), "r"(q + 1) : "memory");
          if (++a >= kASlots) {
            a = 0;
            ph ^= 1;
          }
        }
      }
      PROBE_PRINT("A producer");
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------ MMA issuer
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
    // The whole warp runs the loop (warp-uniform control flow and addresses: the compiler keeps them in uniform registers);
    // one elected lane issues.  A: tensor memory, lane = row of the tile, 8 columns per K step (re of shots 4j .. 4j+3 | im of
    // the same shots), hi at column 16 j of the stage's slot, lo at 16 j + 8.  B: MN-major tf32 must use the 128-byte swizzle
    // with 32-byte atoms (the only MN-major layout the tensor core takes for 32-bit operands): a region is [nblk blocks of
    // 32 columns][8 shot rows][128 B]; LBO = 1024 (next column block); the K step's first four rows are shots 4j .. 4j+3 of
    // B0 (512 j into the block), its second four rows sit SBO = 2 regions further: the same shots of B1 = i B0.
    const uint32_t base16 = (smem_u32(planes) & 0x3FFFF) >> 4, stage16 = PLANES >> 4;
    const uint32_t hiB = ((2 * REG) >> 4) | (1u << 14) | (LAYOUT_SW128_BASE32B << 29);
    const uint32_t loB_hi0 = base16 | ((BLK_BYTES >> 4) << 16), loB_lo0 = loB_hi0 + (REG >> 4);  // (K step 1: + 32)
    const uint32_t tmA0 = tmem_base + kTmemA;
    uint32_t g = 0, it = 0;  // global chunk index; global stage index
    PROBE_DECL;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
      const int rem = t % per_bin, ni = rem % P.ntl;
      const uint32_t idesc = instr_desc((uint32_t)(tile_col0(P, ni + 1) - tile_col0(P, ni)));  // a multiple of 32, <= BN
      for (int kb0 = 0; kb0 < KB; kb0 += kChunk, ++g) {
        const int b = g & 1;
        if (g >= 2) PROBE_WAIT(0, flag_wait_ge(drained + b, kReadWarps * (g >> 1)));  // every earlier chunk of this buffer has been read out
        const uint32_t d = tmem_base + (uint32_t)b * BN;
        const int kb1 = min(kb0 + kChunk, KB);
        for (int kb = kb0; kb < kb1; ++kb) {
          const uint32_t s = it & (kTmemSlots - 1);
          PROBE_WAIT(1, flag_wait_ge(ready + s, (it >> kLgSlots) + 1));
          __syncwarp();  // the lanes leave the polling loop one by one: elect.sync needs them all back
          tc_fence_after();
          const uint32_t off = s * stage16, ta = tmA0 + s * kTmemAStage;
          if (elect_one()) {
            // small terms first; a chunk starts from zero
            if (!(P.tune & 8)) {
#pragma unroll
              for (int h = 0; h < kSub; ++h) {
                const uint32_t o = off + h * (SUBPL >> 4), a = ta + 32 * h;
                umma_tf32_ts(d, a + 8, loB_hi0 + o, hiB, idesc, kb != kb0 || h != 0);
                umma_tf32_ts(d, a, loB_lo0 + o, hiB, idesc, 1);
                umma_tf32_ts(d, a, loB_hi0 + o, hiB, idesc, 1);
                umma_tf32_ts(d, a + 24, loB_hi0 + o + 32, hiB, idesc, 1);
                umma_tf32_ts(d, a + 16, loB_lo0 + o + 32, hiB, idesc, 1);
                umma_tf32_ts(d, a + 16, loB_hi0 + o + 32, hiB, idesc, 1);
              }
            }
            umma_commit(empty + s);
          }
          __syncwarp();
          ++it;
        }
        if (elect_one()) umma_commit(acc_full + b);
        __syncwarp();
      }
    }
    if (lane == 0) PROBE_PRINT("MMA issuer");
  } else if (warp == 2) {
    // ------------------------------------------------------------------------------------ relay
    // Readiness of a stage reaches the MMA warp through a shared-memory word, not through the mbarrier (header).  The
    // split warps cannot write that word themselves: a plain store could become visible before their proxy fence has
    // taken effect (measured: with a fast issuer the tensor core then read stale operands), whereas an mbarrier arrive is
    // ordered behind the fence.  So they arrive on split_bar and this thread turns the completed phase into the word.
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
    if (lane == 0) {
      uint32_t it = 0;
      PROBE_DECL;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x)
        for (int kb = 0; kb < KB; ++kb, ++it) {
          const uint32_t s = it & (kTmemSlots - 1);
          PROBE_WAIT(0, mbar_wait(split_bar + s, (it >> kLgSlots) & 1));
          flag_set(ready + s, (it >> kLgSlots) + 1);
        }
      PROBE_PRINT("relay");
    }
  } else if (warp == 3) {
    // ------------------------------------------------------------------------------------ TMA producer of the B tiles
    // (a thread issues one TMA instruction per ~250 clk and an expect_tx per ~150, measured: with both tiles on one
    // thread the producer alone needed ~850 clk per stage, more than the stage's MMAs)
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      PROBE_DECL;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int kk = t / per_bin, rem = t - kk * per_bin, ni = rem % P.ntl;
        for (int kb = 0; kb < KB; ++kb) {
          PROBE_WAIT(0, mbar_wait(emptyB + s, ph ^ 1));
          if (P.tune & (64 | 256)) {
            mbar_arrive(fullB + s);
          } else {
            mbar_expect_tx(fullB + s, RAW);
            // eight dense rows of nblk x 128 bytes (8 rows for the TMA unit instead of 8 nblk in the tensor core's layout);
            // columns past 2 ldf arrive as zeros (and still count their bytes)
            tma_load_2d(&tmB, fullB + s, rawB + (size_t)s * RAW, tile_col0(P, ni), kk * P.ld + kb * BKC * kSub);
          }
          if (++s == NRB) {
            s = 0;
            ph ^= 1;
          }
        }
      }
      PROBE_PRINT("B producer");
    }
  } else if (warp < kFirstReadWarp) {
    // ------------------------------------------------------------------------------------ split warps
    // Three groups of four warps; group g takes the stages g, g + 3, g + 6, ... of this CTA's stage sequence, so the
    // latency chain of one stage (waits, LDS -> ALU -> STS / tcgen05.st, fences, arrive: ~1400 clk measured, against 576 clk
    // of MMAs per stage) overlaps the other groups'.
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsSplit));
    const int grp = (warp - 4) / kSplitWarps;
    const int wt = threadIdx.x - 128 - grp * kSplitThreads;  // 0 .. 127
    const uint32_t planes_base = smem_u32(planes), raw_base = smem_u32(rawB), a_base = smem_u32(smem);
    // A: this thread owns row ar = 32 (warp % 4) + lane of the tile (the TMEM lanes its warp may write) and reads the 64 bytes
    // of the stage's half of the box (stage it = half it % 2 of box it / 2): K step j = bytes 32 j .. 32 j + 31 of the half =
    // (re0 im0 re1 im1 | re2 im2 re3 im3) of shots 4 j .. 4 j + 3.  SWIZZLE_128B: the 16-byte chunk c of row r sits at
    // chunk position c ^ (r & 7); the second half's chunks (4 + c) sit 64 bytes "xor-away" from the first half's.
    const int ar = 32 * (warp & 3) + lane;
    uint32_t a_off[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) a_off[c] = (uint32_t)ar * 128 + (uint32_t)((c ^ (ar & 7)) << 4);
    const uint32_t a_tmem = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + kTmemA;
    // B: this thread's float4s of the raw tile [8 shots][nblk x 128 B]: q = wt, wt + 128, ... < 8 x 8 nblk; shot row
    // r = q / (8 nblk), column block b and 16-byte chunk c of the block from q % (8 nblk).  In the tensor core's layout the
    // 32-byte unit u of row r of a block sits at unit position u ^ (r & 3) (SWIZZLE_128B with 32-byte atoms).
    const uint32_t per_row = 8 * (uint32_t)P.nblk, nq = 8 * per_row;  // nq <= 384: at most three float4s per thread
    uint32_t b_dst[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const uint32_t q = (uint32_t)wt + i * kSplitThreads, r = q / per_row, x = q - r * per_row, blk = x >> 3, ch = x & 7;
      b_dst[i] = blk * BLK_BYTES + r * 128 + ((((ch >> 1) ^ (r & 3)) << 5) | ((ch & 1) << 4));
    }
    const int nmine = (int)wt < (int)nq ? (int)((nq - wt + kSplitThreads - 1) / kSplitThreads) : 0;
    const int my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const uint32_t total = (uint32_t)my_tiles * (uint32_t)KB;  // stages this CTA runs through
    int rb = grp % NRB;  // slot of stage it in the raw B ring and its phase
    uint32_t phb = (grp / NRB) & 1;
    // kALdg: this thread's receiver row of the current tile, and the stage's position in the tile
    int tile_i = grp / KB, kb = grp % KB, tile_seen = -1;
    const float4* a_row = nullptr;
    static_assert(!(kALdg && kSub == 2), "direct global loads of A exist for 8-shot stages only");
    PROBE_DECL;
    for (uint32_t it = grp; it < total; it += kSplitGroups) {
      // 8-shot stages: stage it is half it % 2 of box it / 2; 16-shot stages: stage it is box it
      const uint32_t box = kSub == 2 ? it : it >> 1, half0 = kSub == 2 ? 0u : (it & 1) << 6;
      const int sa = kALdg ? 0 : (int)(box % (kASlots ? kASlots : 1));  // slot of the raw A box of stage it, and its phase
      const uint32_t pha = kALdg ? 0 : (box / (kASlots ? kASlots : 1)) & 1;
      float4 c[4];
      if (kALdg) {
        if (tile_i != tile_seen) {
          tile_seen = tile_i;
          const int t = blockIdx.x + tile_i * gridDim.x, kk = t / per_bin, mi = (t - kk * per_bin) / P.ntl, r = mi * BM + ar;
          a_row = r < P.n ? P.Rhat4 + (size_t)r * P.a_row4 + (size_t)kk * P.ld4 : nullptr;  // rows past the last receiver are zeros
        }
        if (a_row) {
#pragma unroll
          for (int k = 0; k < 4; ++k) c[k] = ldg128_stream(a_row + 4 * kb + k);
        } else {
#pragma unroll
          for (int k = 0; k < 4; ++k) c[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        kb += kSplitGroups;
        while (kb >= KB) {
          kb -= KB;
          ++tile_i;
        }
      }
      const uint32_t s = it & (kTmemSlots - 1);  // operand stage: B planes in shared memory, A slot in tensor memory
      if (P.tune & 32) {
        mbar_wait(fullB + rb, phb);
        if (!kALdg) mbar_wait(fullA + sa, pha);
        if (it >= kTmemSlots) mbar_wait(empty + s, ((it >> kLgSlots) - 1) & 1);
        __syncwarp();
        if (lane == 0) {
          if (!kALdg) mbar_arrive(emptyA + sa);
          mbar_arrive(emptyB + rb);
          mbar_arrive(split_bar + s);
        }
      } else {
#if MK_TC_TEST2
      // The raw rings run stages ahead, so both tiles are normally long there - but a wait costs ~150 clk even then: the two
      // are asked in one go (independent instructions, their latencies overlap); only a tile that is really missing is waited for.
      {
        const uint32_t okA = kALdg ? 1u : mbar_test(fullA + sa, pha), okB = mbar_test(fullB + rb, phb);
        if (!okA) PROBE_WAIT(0, mbar_wait_warp(fullA + sa, pha));
        if (!okB) PROBE_WAIT(1, mbar_wait_warp(fullB + rb, phb));
      }
#else
      if (!kALdg) PROBE_WAIT(0, mbar_wait_warp(fullA + sa, pha));
      PROBE_WAIT(1, mbar_wait_warp(fullB + rb, phb));
#endif
      const uint32_t raw = raw_base + (uint32_t)rb * RAW, st = planes_base + s * PLANES, ta = a_tmem + s * kTmemAStage;
#pragma unroll
      for (int h = 0; h < kSub; ++h) {  // the 8-shot sub-stages of the stage
        if (!kALdg) {
#pragma unroll
          for (int k = 0; k < 4; ++k) c[k] = lds128(a_base + (uint32_t)sa * A_BOX_BYTES + (a_off[k] ^ (half0 | ((uint32_t)h << 6))));
        }
        float4 v[3];
#pragma unroll
        for (int i = 0; i < 3; ++i)
          if (i < nmine) v[i] = lds128(raw + h * REG + (((uint32_t)wt + i * kSplitThreads) << 4));
        // The operand stage (B planes, A slot) is free once the MMAs of stage it - 4 have retired: empty[s] cannot run a
        // second phase ahead, its next completion belongs to stage it itself.
        if (h == 0 && it >= kTmemSlots) {
          PROBE_WAIT(2, mbar_wait_warp(empty + s, ((it >> kLgSlots) - 1) & 1));
          tc_fence_after();
        }
        // B: raw tile -> B0_hi (copy), B0_lo, and B1 = i B0 (every float4 holds two (re, im) pairs) hi / lo
#pragma unroll
        for (int i = 0; i < 3; ++i)
          if (i < nmine && !(P.tune & 16)) {
            const uint32_t dst = st + h * SUBPL + b_dst[i];
            const float4 l = lo4(v[i]);
            sts128(dst, v[i]);
            sts128(dst + REG, l);
            sts128(dst + 2 * REG, make_float4(-v[i].y, v[i].x, -v[i].w, v[i].z));
            sts128(dst + 3 * REG, make_float4(-l.y, l.x, -l.w, l.z));
          }
        // A -> tensor memory: per K step hi (re0 re1 re2 re3 | im0 im1 im2 im3), lo beside it
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const float4 re = make_float4(c[2 * j].x, c[2 * j].z, c[2 * j + 1].x, c[2 * j + 1].z),
                       im = make_float4(c[2 * j].y, c[2 * j].w, c[2 * j + 1].y, c[2 * j + 1].w);
          tmem_st16(ta + 32 * h + 16 * j, re, im, lo4(re), lo4(im));
        }
      }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the tensor core
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (!kALdg) mbar_arrive(emptyA + sa);  // this warp's part of the raw tiles is in registers / tensor memory / the planes
        mbar_arrive(emptyB + rb);
        mbar_arrive(split_bar + s);
      }
      }
      rb += kSplitGroups;
      while (rb >= NRB) {
        rb -= NRB;
        phb ^= 1;
      }
    }
    if (wt == 0) PROBE_PRINT(grp == 0 ? "split g0" : (grp == 1 ? "split g1" : "split g2+"));
  } else {
    // ------------------------------------------------------------------------------------ read-out warps: chunk sums in registers
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsRead));
    const int quad = warp & 3;         // TMEM lanes 32 quad .. 32 quad + 31 are the ones this warp may read
    const int half = (warp - kFirstReadWarp) >> 2;  // columns (BN / 2) half .. + BN / 2 - 1 of the tile
    uint32_t g = 0;
    PROBE_DECL;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
      const int kk = t / per_bin, rem = t - kk * per_bin, mi = rem / P.ntl, ni = rem - mi * P.ntl;
      const int col0 = tile_col0(P, ni);
      const int cols = tile_col0(P, ni + 1) - col0 - half * (BN / 2);  // valid columns of this warp's half (may exceed BN / 2, may be <= 0)
      float sum[BN / 2];
#pragma unroll
      for (int i = 0; i < BN / 2; ++i) sum[i] = 0.f;
      for (int kb0 = 0; kb0 < KB; kb0 += kChunk, ++g) {
        const int b = g & 1;
        PROBE_WAIT(0, mbar_wait_warp(acc_full + b, (g >> 1) & 1));
        tc_fence_after();
        const uint32_t ta = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(b * BN + half * (BN / 2));
#if MK_TC_READ16   // (two such loads in flight per wait spill in the 128-register budget: 331 us / 1684 us, slower)
#pragma unroll
        for (int c = 0; c < BN / 32; ++c) {
          if (c * 16 < cols && !(P.tune & 4)) {  // warp-uniform (the MMA's N is a multiple of 32); columns past it hold stale data
            uint32_t v[16];
            tmem_ld16(ta + (uint32_t)(c * 16), v);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int q = 0; q < 16; ++q) sum[c * 16 + q] += __uint_as_float(v[q]);
          }
        }
#else
#pragma unroll
        for (int c = 0; c < BN / 16; ++c) {
          if (c * 8 < cols && !(P.tune & 4)) {  // warp-uniform; columns past the MMA's N hold stale data
            uint32_t v[8];
            tmem_ld8(ta + (uint32_t)(c * 8), v);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int q = 0; q < 8; ++q) sum[c * 8 + q] += __uint_as_float(v[q]);
          }
        }
#endif
        tc_fence_before();
        __syncwarp();
        if (lane == 0) flag_add(drained + b);
      }
      const int r = mi * BM + quad * 32 + lane;
      if (r < P.n) {
        float* dst = Shat + (size_t)r * P.s_row + (size_t)kk * P.ncols + col0 + half * (BN / 2);
#pragma unroll
        for (int q = 0; q < BN / 8; ++q)
          if (q * 4 < cols)
            *reinterpret_cast<float4*>(dst + q * 4) = make_float4(sum[4 * q], sum[4 * q + 1], sum[4 * q + 2], sum[4 * q + 3]);
      }
    }
    if (warp == kFirstReadWarp && lane == 0) PROBE_PRINT("read-out w0");
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

int encode(mk_ctx* c, EncodeTiledFn enc, void* out, const void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
           const cuuint32_t* box, CUtensorMapSwizzle sw, const char* what) {
  const cuuint32_t es[3] = {1, 1, 1};
  const CUresult r = enc(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, (cuuint32_t)rank, const_cast<void*>(base), dims,
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
  int major = 0;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, c->dev);
  return major == 10 && c->smem_optin >= fixed_smem(1) + 2 * kSub * BLK_BYTES + kSmemExtra;
}

int launch_syn_tc(mk_ctx* c, const RowBlock& rb, int slot, const float2* d_Nhat, float2* d_Shat, int ldf) {
  if (ldf % 16 != 0) return set_err(c, MK_ERR_INVALID_ARG, "the tcgen05 contraction needs ldf to be a multiple of 16");
  EncodeTiledFn enc = nullptr;
  if (int rc = get_encode(c, &enc)) return rc;
  // descriptor cache: the resident rows, or one of the two streaming windows (mk_create_streamed)
  const int ia = rb.Rhat == c->d_win[0] && c->d_win[0] ? 1 : (rb.Rhat == c->d_win[1] && c->d_win[1] ? 2 : 0);
  if (c->tmap_A_key[ia] != rb.Rhat || c->tmap_A_rows[ia] != rb.nrow) {
    // A = R^ as fp32 [n][nb][2 ld]: dims (float of the row, bin, r); box = 32 floats (16 shots) x 1 bin x 128 receivers; rows r >= n read as zero
    const cuuint64_t dims[3] = {(cuuint64_t)2 * c->ld, (cuuint64_t)c->nb, (cuuint64_t)rb.nrow};  // rows of this block
    const cuuint64_t str[2] = {(cuuint64_t)2 * c->ld * 4, (cuuint64_t)c->nb * 2 * c->ld * 4};
    const cuuint32_t box[3] = {4 * BKC, 1, BM};
    if (int rc = encode(c, enc, c->tmap_A[ia], rb.Rhat, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, "A")) return rc;
    c->tmap_A_key[ia] = rb.Rhat;
    c->tmap_A_rows[ia] = rb.nrow;
  }
  const int nblk = std::min(BN / 32, (2 * ldf) / 32);
  if (c->tmap_B_key[slot] != d_Nhat || c->tmap_B_ldf[slot] != ldf) {
    // B = N^ as fp32 [nb * ld rows][2 ldf floats]: box = nblk x 32 floats of 8 consecutive rows (shots), dense in shared
    // memory; the split warps put it into the tensor core's MN-major layout
    const cuuint64_t dims[2] = {(cuuint64_t)2 * ldf, (cuuint64_t)c->nb * c->ld};
    const cuuint64_t str[1] = {(cuuint64_t)2 * ldf * 4};
    const cuuint32_t box[2] = {(cuuint32_t)nblk * 32, BKC * kSub};  // nblk is a function of ldf: one cache key
    if (int rc = encode(c, enc, c->tmap_B[slot], d_Nhat, 2, dims, str, box, CU_TENSOR_MAP_SWIZZLE_NONE, "B")) return rc;
    c->tmap_B_key[slot] = d_Nhat;
    c->tmap_B_ldf[slot] = ldf;
  }
  TcParams P;
  P.n = rb.nrow;  // rows of this block; S^ is offset to the first one below
  P.nb = c->nb;
  P.ld = c->ld;
  P.ncols = 2 * ldf;
  P.mt = (rb.nrow + BM - 1) / BM;
  P.ntl = (P.ncols + BN - 1) / BN;
  P.nblocks = P.ncols / 32;
  P.Rhat4 = reinterpret_cast<const float4*>(rb.Rhat);
  P.a_row4 = (size_t)c->nb * c->ld / 2;
  P.ld4 = c->ld / 2;
  P.a_tiled = c->rhat_layout == 1;
  P.s_row = (size_t)c->nb * 2 * ldf;
  P.nblk = nblk;
  P.tune = c->tune;
  const size_t raw_b = (size_t)kSub * nblk * BLK_BYTES;
  if (c->smem_optin < fixed_smem(nblk) + kSmemExtra + 2 * raw_b)
    return set_err(c, MK_ERR_INVALID_ARG, "not enough shared memory for the tcgen05 contraction");
  // what is left after the operand stages goes to the raw rings: 6 B tiles first, then A boxes (the deeper ring: R^ comes
  // from HBM or L2 at the rate the bytes in flight allow), then up to 8 B tiles
  size_t left = c->smem_optin - kSmemExtra - fixed_smem(nblk);
  P.nrb = (int)std::min<size_t>(6, left / raw_b);
  left -= P.nrb * raw_b;
  P.na = kMinASlots + (kALdg ? 0 : (int)std::min<size_t>(kMaxASlots - kMinASlots, left / A_BOX_BYTES));
  left -= (size_t)(P.na - kMinASlots) * A_BOX_BYTES;
  P.nrb += (int)std::min<size_t>(kMaxRawB - P.nrb, left / raw_b);
  if (c->tune & 512) {
    P.nrb = std::min(P.nrb, 3);
    P.na = kMinASlots;
  }
  const size_t kSmemBytes = (size_t)P.na * A_BOX_BYTES + kTmemSlots * (size_t)planes_bytes(nblk) + (size_t)P.nrb * raw_b + kSmemExtra;
  const int ntiles = P.nb * P.mt * P.ntl;
  // (in step: a multiple of ntl, so that every CTA keeps its N tile and its siblings, see the A producer)
  const bool in_step = (c->tune & 1024) && P.ntl > 1 && P.ntl <= c->num_sms;  // measurement switch, off: it costs more than it saves
  const int grid = ntiles < c->num_sms ? ntiles : (in_step ? (c->num_sms / P.ntl) * P.ntl : c->num_sms);
  P.progress = nullptr;
  if (in_step && grid % P.ntl == 0 && grid <= 1024) {
    if (!c->d_tc_progress)
      if (int rc = check_cuda(c, cudaMalloc(&c->d_tc_progress, 1024 * sizeof(uint32_t)), "cudaMalloc progress")) return rc;
    if (int rc = check_cuda(c, cudaMemsetAsync(c->d_tc_progress, 0, 1024 * sizeof(uint32_t), c->stream), "memset progress")) return rc;
    P.progress = c->d_tc_progress;
  }
  float* S0 = reinterpret_cast<float*>(d_Shat + (size_t)rb.r0 * c->nb * ldf);
  const CUtensorMap& mA = *reinterpret_cast<const CUtensorMap*>(c->tmap_A[ia]);
  const CUtensorMap& mB = *reinterpret_cast<const CUtensorMap*>(c->tmap_B[slot]);
  if (int rc = check_cuda(c, cudaFuncSetAttribute(k_syn_gemm_tf32x3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes), "cudaFuncSetAttribute"))
    return rc;
  k_syn_gemm_tf32x3<<<grid, kThreads, kSmemBytes, c->stream>>>(mA, mB, S0, P);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_syn_gemm_tf32x3");
}

}  // namespace mk
