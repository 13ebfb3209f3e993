/* mk.h — C ABI of libmk: the synthesis hot path of the iterative Neumann-series Marchenko method
 * (arXiv 2106.04649) as hand-written sm_100a CUDA kernels.  One GPU, one context per reflection response.
 *
 * Citations: "PAPER.md:N" = /root/reference/PAPER.md line N; "§8" = SURVEY.md section 8; G1..G14 = the
 * readings of the paper listed in DESIGN.md.
 *
 * What the library computes (notation of §8):
 *   nshot sources, nrec receivers (n = nshot = nrec for a co-located fixed spread, as in every BASELINE.json config; see
 *   mk_set_geometry for the general case); time index j in [0, nt), negative times stored wrapped
 *   (T f)[j] = f[(nt - j) % nt];  band B = {klo..khi} = {k : fmin <= k/(nt dt) <= fmax};  w[s] trapezoid weights
 *   synthesis  (R N)[f][r][j] = P_B { dt * sum_s w[s] * sum_j' R[s][r][(j - j') % nt] * N[f][s][j'] }      eq. (1)
 *   window     Theta[f][r][j] = ( |j+-| < h ),  h = clamp(floor(t_d/dt + 0.5) - eps, 0, nt/2)               PAPER.md:24, G2
 *   one step   N_i = - Theta T R N_{i-1},   N_{-1} = T G_d
 *   f1plus = N_{-1} + sum_{i odd} N_i ;  f1min = - sum_{i even} T N_i ;  p^- = sum_i R N_{i-1}
 *   G^- = R f1plus - f1min ;  G^+ = T f1plus - R (T f1min) ;  G = p^- + T f1plus - f1min                    PAPER.md:24, 87-88, G3-G5
 * The time convolution runs in the frequency domain: per bin k in B a complex contraction of
 * R^[r][k][s] over source positions s against N^[s][k][f] — a streaming GEMV for few focal points, a batched
 * complex GEMM for many.
 *
 * Conventions for every entry point
 *   - returns int: MK_OK (0) or a negative MK_ERR_* code; never throws or aborts across the ABI;
 *     mk_last_error(ctx) returns a NUL-terminated description of the last failure on that context.
 *   - "d_" arguments are DEVICE pointers owned by the caller (allocated e.g. with PyTorch), 16-byte aligned;
 *     "h_" arguments are HOST pointers owned by the caller (pinned memory makes the copies asynchronous).
 *     The library never frees or retains caller buffers beyond the call (work is stream-ordered: a d_ buffer
 *     may be reused once the context's stream has reached the end of the call).
 *   - the library owns R^ (band-limited complex64 reflection response), its accumulators and workspaces.
 *   - all work is enqueued on the context's stream (the legacy default stream until mk_set_stream).
 *     d_-pointer calls do not synchronise the host; h_-pointer calls return after the results are in host memory.
 *   - there is no CPU fallback: without a CUDA device mk_create fails with MK_ERR_CUDA.
 *   - a context lives on the CUDA device that was current in mk_create; every entry point makes that device current
 *     again (cudaSetDevice) before it does anything, so the caller may switch devices between calls.
 *   - run state: mk_begin / mk_run start a run; mk_step, mk_finish*, mk_image, mk_operand need one.  Calls that change
 *     what the run was started from — mk_load_R (another R^), MK_OPT_EPS_SAMPLES with a new value (another window),
 *     mk_operand_reserve with another nfoc / regime (another operand layout) — END the run: afterwards the calls that
 *     need a run return MK_ERR_STATE until the next mk_begin / mk_run.  Between mk_step_contract and mk_step_post they
 *     are refused with MK_ERR_STATE.  MK_OPT_REGIME only affects runs started afterwards (a run keeps its regime);
 *     mk_synthesis picks its own regime from its own nfoc and never disturbs the run in progress.
 */
#ifndef MK_H_
#define MK_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mk_ctx mk_ctx; /* opaque */

enum {
  MK_OK = 0,
  MK_ERR_INVALID_ARG = -1, /* NULL pointer, non-positive size, nshot != nrec, nt not a power of two, ... */
  MK_ERR_STATE = -2,       /* mk_run before every shot was loaded, mk_step before mk_begin, ... */
  MK_ERR_OOM = -3,         /* device allocation failed */
  MK_ERR_CUDA = -4         /* a CUDA call failed (sticky; text in mk_last_error) */
};

/* mk_set_option keys */
enum {
  MK_OPT_EPS_SAMPLES = 1, /* window margin eps in samples (default 8; BASELINE.json config 0; G2) */
  MK_OPT_REGIME = 2,      /* contraction kernel: 0 auto (default: 1 for nfoc <= 8, else 3), 1 streaming GEMV,
                             2 FP32-FFMA GEMM, 3 tcgen05 3xTF32 GEMM with chunked fp32 accumulation (sm_100 only;
                             MK_ERR_INVALID_ARG otherwise).  Affects runs / syntheses started afterwards */
  MK_OPT_TIMING = 3,      /* N >= 1: bracket every N-th contraction launch with CUDA events on the context's stream (1: every
                             one; a record between two kernels costs ~3 us and keeps them from overlapping, so a sparse
                             sample disturbs a step of many short launches less); 0: off */
  MK_OPT_FUSED_FINALS = 5, /* 1 (default): with 1, 2 or 4 focal points mk_finish / mk_run compute the extra syntheses of G^- and
                             G^+ in ONE pass over R^ (2 nfoc right-hand sides, streaming GEMV); 0: one pass each */
  MK_OPT_FFT_PATH = 4,    /* transform kernels: 0 auto (default), 1 generic shared-memory passes (any nt),
                             2 register-resident path (nt = 2048 or 4096 only; MK_ERR_INVALID_ARG otherwise) */
  MK_OPT_RHAT_FORMAT = 6, /* NEXT-4 (compressed R "accelerates data loading"): storage of
                             R^.  0 (default): complex64.  1: "q16" block floating point — per (receiver, bin) row, blocks of
                             16 shots share one fp32 scale sc = max(|re|, |im|) / 32767 and every component is the int16
                             rint(v / sc): 4.25 bytes per complex element instead of 8, error <= sc / 2 per component.  The
                             lossy format serves the bandwidth-bound regime only (nfoc <= 8, streaming GEMV with fp32
                             accumulation; more focal points: MK_ERR_INVALID_ARG) and is held to its own tolerance
                             (DESIGN.md section 6c), not to north_star's.  Must be set before the first mk_load_R
                             (MK_ERR_STATE afterwards); with it mk_load_R needs shot0 and nshots to be multiples of 16
                             (except at the last shot).  Not available on row-sharded or streamed contexts */
  MK_OPT_RHAT_LAYOUT = 8, /* memory layout of R^ in HBM.  0 (default): [rec][bin][shot], one (receiver, bin) row contiguous —
                             what the streaming GEMV reads; every regime works on it.  1: TILED for the tensor regime:
                             [rec / 128][bin][shot / 16] boxes of [128 receivers][16 shots] = 16 KB contiguous (receiver rows
                             padded to a multiple of 128), the unit the tcgen05 contraction consumes per two stages, fetched
                             with ONE bulk copy instead of 128 rows 2 MB apart.  Only the tcgen05 regime reads it (every nfoc
                             then takes regime 3; MK_OPT_REGIME 1 / 2: MK_ERR_INVALID_ARG).  Must be set before the first
                             mk_load_R (MK_ERR_STATE afterwards); plain contexts only (not sharded / streamed / compressed) */
  MK_OPT_TUNE = 7         /* measurement switches, a bit mask (default 0 = the product path).  bit 0: k_post_fast does not
                             prefetch the next tile's spectra to L2 (same results).  Bits 2..5 leave out one part of the
                             tcgen05 contraction to find what bounds it; the RESULTS ARE WRONG with any of them: 4 = the
                             read-out warps do not read tensor memory, 8 = no MMA is issued, 16 = the split warps skip the
                             B planes, 32 = the split warps do nothing, 64 = no TMA load is issued,
                             128 = no A tile is loaded, 256 = no B tile is loaded.  512: the raw B ring has 3 slots; 1024: the CTAs
                             that share an A tile keep in step through global progress counters (same results, slower); 2048: the
                             fused pass of nt = 4096 takes eight traces per CTA (512 threads, one CTA per SM) instead of four
                             (same results, same speed); 4096: no kernel is launched with programmatic dependent launch
                             (same results; the launch gaps of the short kernels come back: +0.01 .. 0.04 ms per config-1 step);
                             8192: the kernels do nothing ahead of griddepcontrol.wait (no twiddle tables pulled into L1 by the
                             few-trace FFT kernels, no L2 prefetch of the first rows of R^ by the streaming GEMV; same results) */
};

/* mk_get_info keys (values returned as double) */
enum {
  MK_INFO_NB = 1,            /* number of bins in B */
  MK_INFO_KLO = 2,           /* first bin of B */
  MK_INFO_KHI = 3,           /* last bin of B */
  MK_INFO_RHAT_BYTES = 4,    /* algorithmic bytes of R^: 8 * nrec * nb * nshot (unpadded) */
  MK_INFO_RHAT_BYTES_PADDED = 5,
  MK_INFO_LD_SHOT = 6,       /* padded shot dimension of R^ (multiple of 16 elements = 128 B) */
  MK_INFO_SHOTS_LOADED = 7,
  MK_INFO_SYN_LAUNCHES = 8,  /* contraction launches timed since the last MK_INFO_SYN_RESET (needs MK_OPT_TIMING) */
  MK_INFO_SYN_MS_TOTAL = 9,  /* their summed device time in ms (synchronises the stream) */
  MK_INFO_SYN_RESET = 10,    /* resets the two counters above; value returned is 0 */
  MK_INFO_KERNEL_LAUNCHES = 11, /* total kernels this context has launched since creation */
  MK_INFO_REGIME_USED = 12,  /* regime of the last contraction launch (1, 2 or 3) */
  MK_INFO_DEVICE_BYTES = 13, /* device memory currently owned by the context */
  MK_INFO_RESIDENT_ROWS = 14, /* rows of R^ kept in HBM (== rows owned unless mk_create_streamed) */
  MK_INFO_WINDOW_ROWS = 15,  /* rows per streaming window (0: R^ is resident) */
  MK_INFO_H2D_BYTES = 16,    /* bytes of R^ the contractions have copied host -> device since mk_create_streamed */
  MK_INFO_RHAT_BYTES_STORED = 17, /* bytes R^ occupies as stored (padded): 8 per element, 4.25 with MK_OPT_RHAT_FORMAT = 1 */
  MK_INFO_RHAT_LAYOUT = 18,  /* MK_OPT_RHAT_LAYOUT as set */
  MK_INFO_SYN_COUNT = 19     /* contraction launches since the last MK_INFO_SYN_RESET, timed or not */
};

/* Create a context for an nshot x nrec x nt reflection response sampled at dt (s) and dx (m), band fmin..fmax (Hz).
 * Validates nshot, nrec > 0, nt a power of two in [16, 32768], dt, dx > 0, 0 <= fmin <= fmax <= 1/(2 dt).  With
 * nshot == nrec the spread is taken as co-located (shot s at receiver s: the output index of one iteration is the
 * integration index of the next, G10); otherwise see mk_set_geometry.
 * Allocates R^ [nrec][nb][ld_shot] complex64 on the current CUDA device (BASELINE.json north_star (a)
 * "the data layout is ordered as receivers, frequencies and shots").  *out receives the context; when a failure
 * happens after the context exists, *out is still set so that mk_last_error can be read (destroy it afterwards),
 * otherwise *out is NULL. */
int mk_create(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax);

/* NEXT-3, second half: out-of-core R^ for a reflection response whose band-limited spectrum does not
 * fit the device.  The paper's largest experiment exists for exactly this case ("synthesis must be done in a
 * batched fashion ... a certain batch is transferred to each GPU"; Algorithm 2's copyH2D_shot_batch loop, PAPER.md:98-112;
 * the 249 GB set "forces pipelining").  Rows 0 .. resident_rows-1 of R^ [nrec][nb][ld_shot] stay in HBM;
 * the other rows live in pinned host memory owned by the context (written there directly by the ingest kernel of
 * mk_load_R), and every contraction streams them through two windows of window_rows rows in HBM (0 = choose: 1/8 of the
 * host rows), one cudaMemcpyAsync per row block on a copy stream, overlapped with the contraction of the previous
 * block; passes alternate direction so that the two blocks left in the windows are not transferred again.  Everything
 * else (operands, spectra, time fields, every other call) is as with mk_create; results equal the resident context's
 * bit for bit.  resident_rows in [0, nrec]; resident_rows == nrec is mk_create.  Not combinable with row sharding. */
int mk_create_streamed(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax,
                       int resident_rows, int window_rows);

/* Frees everything the context owns.  NULL is accepted. */
int mk_destroy(mk_ctx* ctx);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = legacy default stream. */
int mk_set_stream(mk_ctx* ctx, void* cuda_stream);

int mk_set_option(mk_ctx* ctx, int key, double value);
int mk_get_info(mk_ctx* ctx, int key, double* value);

/* NEXT-4: sources and receivers that are not co-located one to one, irregular source spacing.
 * Eq. (1) integrates over SOURCE positions and is evaluated at RECEIVER positions (PAPER.md:28 keeps
 * "ns" and "nr" apart): G_d, t_d and every output field live on the receiver grid, [nfoc][nrec][nt]; the operand of the
 * next synthesis lives on the shot grid.  h_rec_of_shot [nshot] (HOST, int): the receiver co-located with shot s, or -1
 * when there is none — that source position then carries a zero operand, it contributes nothing to the integral because
 * the field is not known there (reading G15); two shots may not share a receiver.  NULL = shot s at receiver
 * s (for s < min(nshot, nrec)), which is also the state after mk_create.  h_weights [nshot] (HOST, float): quadrature
 * weights w[s] of the shot grid in metres (finite, >= 0), folded into R^ at ingest; NULL = trapezoid rule with spacing
 * dx.  Must be called before the first mk_load_R (MK_ERR_STATE afterwards) and not on a row-sharded context. */
int mk_set_geometry(mk_ctx* ctx, const int* h_rec_of_shot, const float* h_weights);

/* Ingest ("the whole reflection data being read, Fourier transformed and stored", 63-66; §8(a) a0).
 * d_R_time: [nshots][nrec][nt] fp32 time-domain R(x_R = rec, x = shot, t) for shots shot0 .. shot0+nshots-1.
 * Converted on the GPU, once, to band-limited complex64 with the quadrature weights folded in:
 *   R^[r][k][s] = dt * w[s] * sum_j R[s][r][j] e^{-2 pi i k j / nt},  k in B  (shot index fastest, zero padded to ld_shot).
 * May be called repeatedly with disjoint shot ranges (config 4: 61 calls of 64 shots), and again later to replace
 * shots (it ends a run in progress, see "run state" above). */
int mk_load_R(mk_ctx* ctx, const float* d_R_time, int shot0, int nshots);
/* The same for a source that holds only the receiver rows this context owns: d_R_rows is [nshots][nrows][nt] with
 * nrows = the context's rows (row0 .. row0+nrows-1 of mk_create_sharded; all nrec rows otherwise, where the call equals
 * mk_load_R).  With it the G ranks of a row-sharded run read 1/G of R each instead of all of it (config 4: 250 GB of
 * time-domain R would otherwise be produced G times).  Not available with compressed or out-of-core R^. */
int mk_load_R_rows(mk_ctx* ctx, const float* d_R_rows, int shot0, int nshots);
/* Same as mk_load_R from a HOST buffer: staged through an internal device buffer in bounded chunks; returns when done. */
int mk_load_R_host(mk_ctx* ctx, const float* h_R_time, int shot0, int nshots);

/* Outputs of a run; each pointer is [nfoc][nrec][nt] fp32 or NULL to skip that field.  G^- and G^+ cost one
 * extra synthesis each ("estimating each component requires an extra synthesis"). */
typedef struct mk_outputs {
  float* N_last; /* N_{niter-1}; honoured by mk_run / mk_run_host only (mk_finish rejects it: use mk_step's d_N_i) */
  float* f1plus;
  float* f1min;
  float* G;
  float* Gplus;
  float* Gminus;
} mk_outputs;

/* The whole scheme (Algorithm 1) for nfoc focal points:
 * d_Gd [nfoc][nrec][nt] fp32 first arrivals G_d(x_R, x_F, t), d_td [nfoc][nrec] fp32 traveltimes in seconds.
 * Equals mk_begin + niter x mk_step + mk_finish.  MK_ERR_STATE unless all nshot shots have been loaded.
 * When d_out->f1plus / f1min are given, the series is accumulated in those fields directly (no copy at the end, no
 * library-owned twin): they must not overlap each other or d_Gd, and until the next mk_begin / mk_run the context reads
 * them again for mk_finish and mk_image, so they must stay allocated and unmodified for those calls.  N_last, G, Gplus
 * and Gminus are written while f1plus / f1min are still read: they must not overlap those two (MK_ERR_INVALID_ARG);
 * they MAY share one buffer among themselves (each is complete before the next is written; the last one written wins:
 * order N_last, Gminus, Gplus, G). */
int mk_run(mk_ctx* ctx, const float* d_Gd, const float* d_td, int nfoc, int niter, const mk_outputs* d_out);
/* Same with HOST inputs and HOST outputs (copies in, runs, copies out, synchronises). */
int mk_run_host(mk_ctx* ctx, const float* h_Gd, const float* h_td, int nfoc, int niter, const mk_outputs* h_out);

/* Step access (same arithmetic; used by the parity tests to see every iterate). */
int mk_begin(mk_ctx* ctx, const float* d_Gd, const float* d_td, int nfoc); /* a1: N_{-1} = f1plus = T G_d, f1min = p^- = 0 */
int mk_step(mk_ctx* ctx, float* d_N_i /* optional [nfoc][nrec][nt] copy of the new iterate, or NULL */); /* a2..a6 */
int mk_finish(mk_ctx* ctx, const mk_outputs* d_out); /* a7; may be called more than once with different fields */
/* mk_step in its two halves: the contraction a2 (reads the operand) and the fused pass a3..a6 (writes the operand of the
 * next step).  With peers attached (mk_operand_attach) the second half stores into the peers' operands too, so every rank
 * must have finished its contraction before any rank runs mk_step_post: put the cross-rank barrier between the two. */
int mk_step_contract(mk_ctx* ctx);
int mk_step_post(mk_ctx* ctx, float* d_N_i);

/* One bare synthesis without window (a6 + a2 + a3): d_S_out = R d_N_in, both [nfoc][nrec][nt] fp32 (with a geometry set
 * by mk_set_geometry, d_N_in is on the receiver grid like every iterate: the trace of receiver r is the operand of the
 * shot co-located with it).  Does not disturb a run in progress.  This is the call the GB/s metric times. */
int mk_synthesis(mk_ctx* ctx, const float* d_N_in, float* d_S_out, int nfoc);

/* NEXT-1 (§8(f)): double-focusing image: the zero-time sample of G^- convolved with f1plus and
 * integrated over receivers (trapezoid rule with spacing dx over the nrec receivers),
 *   image[f] = dt * sum_r w[r] sum_j G^-[f][r][(nt-j)%nt] * f1plus[f][r][j].
 * d_Gminus: [nfoc][nrec][nt] fp32 as returned by mk_run / mk_finish for the current run; d_image: [nfoc] fp32. */
int mk_image(mk_ctx* ctx, const float* d_Gminus, float* d_image);

/* The same image for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): this ONE entry point allocates nothing and frees nothing.  The partial sums of the imaging kernels go
 * to a static device array of MK_IMAGE_STATIC_MAX_PARTIALS doubles (128 KB, part of the library image: every GPU that
 * loads the library holds it until the process exits) instead of the context's scratch buffer.
 *   d_Gminus, d_f1plus: [nfoc][nrec][nt] fp32 device inputs (the two fields are passed explicitly; no run is needed, the
 *   context supplies nrec, nt, dt, dx, the device and the stream); d_image: [nfoc] fp32 device output.
 * Same kernels, same grid, same order of summation as mk_image: for the fields of a run the result is bit-identical.
 * Limit: nfoc x (receiver chunks per focal point) partial sums must fit the array.  The grid has fewer than
 * nfoc + 32 x (SM count) of them, so every nfoc <= MK_IMAGE_STATIC_MAX_PARTIALS - 32 x (SM count) fits (nfoc <= 11648 on
 * a 148-SM B200) and no nfoc > MK_IMAGE_STATIC_MAX_PARTIALS does; beyond the limit the call returns MK_ERR_INVALID_ARG
 * with the numbers in mk_last_error and launches nothing (use mk_image).
 * The first call on a device looks the array's device address up (cudaGetSymbolAddress, no allocation); later calls reuse
 * it.  Every call on a device shares the one array, which keeps the previous call's contents: nothing has to start at
 * zero (each partial sum is written before it is read), but two calls that overlap on the GPU (different streams or
 * contexts on one device, without an ordering between them) race on it and give garbage.  Calls on one stream are safe. */
enum { MK_IMAGE_STATIC_MAX_PARTIALS = 16384 };
int mk_image_static(mk_ctx* ctx, const float* d_Gminus, const float* d_f1plus, float* d_image, int nfoc);

/* ---- NEXT-3: receiver-row sharding across GPUs ------------------------------------------
 * The B200 equivalent of the paper's multi-GPU scheme (every output trace depends on one
 * (receiver, focal point) pair): rank g owns the receiver rows row0 .. row0+nrows-1 of R^ (read-only,
 * never moves) and computes a2..a6 for those rows; the ONE exchange step per synthesis is an all-gather of the rows
 * of the operand N^ the ranks have just produced.  The library computes; the caller moves the rows (NCCL all-gather
 * or peer copies) between the calls, in this order:
 *   mk_create_sharded; mk_load_R (same full chunks on every rank: the library keeps its rows only) or mk_load_R_rows
 *   (each rank passes its own receiver rows only);
 *   mk_begin; [exchange slot 0]; niter x { mk_step; [exchange slot 0] };
 *   for G^-, G^+: mk_finish_prepare(field); [exchange slot 1]; mk_finish_complete(field, out);  mk_finish for f1+-, G.
 * "[exchange slot s]" = read mk_operand(ctx, s, &v), make every rank's rows of every plane identical on all ranks,
 * then call mk_operand_exchanged(ctx, s).  A contraction on an operand whose rows were not exchanged fails with
 * MK_ERR_STATE instead of computing on stale rows.  Time-domain fields keep their full [nfoc][nrec][nt] shape; a
 * rank reads and writes only its own receiver rows of them (the other rows of its outputs are zero or untouched).
 * mk_run, mk_run_host, mk_synthesis and the G^-/G^+ fields of mk_finish need the whole operand at once and return
 * MK_ERR_STATE on a sharded context. */
/* (row sharding exchanges operand rows by receiver index, so a sharded context needs nshot == nrec.) */
int mk_create_sharded(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax,
                      int row0, int nrows);

/* Where the operand of slot 0 (the run) or 1 (finals) lives.  plane[0] is a device array [nb][rows_per_bin][row_floats]
 * fp32: the complex operand N^[k][s][f] as interleaved (re, im) floats, one row per source position (rows_per_rec = 1,
 * rows_per_bin = ld_shot, row_floats = 2 ldf with ldf = nfoc padded to the regime's granularity: 1 / 4 / 16 focal points
 * for regimes 1 / 2 / 3).  Every regime reads this one plane (nplanes = 1; plane[1] is unused and NULL).
 * Valid after mk_begin (slot 0) / mk_finish_prepare (slot 1). */
typedef struct mk_operand_view {
  float* plane[2];
  int nplanes, nb, rows_per_bin, rows_per_rec, row_floats, row0, nrows;
} mk_operand_view;
int mk_operand(mk_ctx* ctx, int slot, mk_operand_view* out);
int mk_operand_exchanged(mk_ctx* ctx, int slot);

/* The exchange fused into the producing kernels (section 8(e): "fused as peer stores from the FFT kernel's epilogue").
 * mk_operand_reserve allocates and zeroes the operands of both slots for runs with nfoc focal points, so that their
 * addresses exist before mk_begin; mk_operand_attach then registers, for one slot, the same slot's operand of up to 7
 * other ranks (views of identical layout, device pointers valid in this process: other contexts of the process, or
 * peer GPU memory mapped through CUDA IPC / peer access).  From then on every kernel of this context that produces
 * operand rows (mk_begin, mk_step, mk_finish_prepare) stores them into its own operand AND, at the same offsets, into
 * every attached one, so no copy is needed afterwards: the caller only has to make sure that all ranks have finished
 * producing (a barrier across the ranks' streams) before it calls mk_operand_exchanged and the next contraction.
 * npeers = 0 detaches.  The attachment is dropped when the operand layout changes (another nfoc or regime). */
int mk_operand_reserve(mk_ctx* ctx, int nfoc);
int mk_operand_attach(mk_ctx* ctx, int slot, int npeers, const mk_operand_view* peers);

/* Plumbing for one process per GPU: CUDA IPC handles of operand planes (each plane is one device allocation), to be
 * exchanged between the ranks by any host channel (torch.distributed all_gather_object) and opened by the peers.
 * handle: 64 bytes.  A pointer opened here must be closed before the exporting context is destroyed. */
int mk_ipc_export(const void* d_ptr, unsigned char handle[64]);
int mk_ipc_open(const unsigned char handle[64], void** d_ptr);
int mk_ipc_close(void* d_ptr);

/* Stream-ordered barrier between the ranks of a row-sharded run (NEXT-3; the ordering the fused exchange needs, without
 * the host: no cudaStreamSynchronize, no host barrier inside the iteration loop).  Every rank owns a small array of
 * world 32-bit flags in device memory (mk_sync_create allocates and zeroes it; mk_sync_flags returns it so that it can
 * be exported with mk_ipc_export and opened by the other ranks, or handed to other contexts of the same process).
 * mk_sync_attach gives the context the flag arrays of ALL ranks as device pointers valid in this process
 * (d_flags_of_rank[rank] may be NULL: the context's own).  mk_sync_barrier then ENQUEUES on the context's stream: one
 * 32-bit write of the next epoch number into flags[rank] of every other rank (ordered behind all work enqueued so far,
 * peer stores of operand rows included), followed by one wait per other rank until that rank's epoch has arrived in the
 * own array (cuStreamWriteValue32 / cuStreamWaitValue32: the GPU's front end waits, no SM is held, the host does not
 * block).  Work enqueued after it on the stream starts only when every rank has reached the same barrier.  All ranks
 * must call it the same number of times.  MK_ERR_CUDA if the driver has no stream memory operations. */
int mk_sync_create(mk_ctx* ctx, int rank, int world);
int mk_sync_flags(mk_ctx* ctx, void** d_flags);
int mk_sync_attach(mk_ctx* ctx, void* const* d_flags_of_rank);
int mk_sync_barrier(mk_ctx* ctx);

enum { MK_FIELD_GMINUS = 1, MK_FIELD_GPLUS = 2 };
int mk_finish_prepare(mk_ctx* ctx, int field);                   /* forward transform of f1plus / T f1min -> slot 1 */
int mk_finish_complete(mk_ctx* ctx, int field, float* d_out);    /* contraction + inverse transform + epilogue      */

const char* mk_last_error(mk_ctx* ctx);
const char* mk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MK_H_ */
