// marchenko_oracle.cpp — TEST INFRASTRUCTURE ONLY (never on the product path).
//
// Plain, slow, double-precision CPU statement of what the synthesis hot path of the iterative
// Neumann-series Marchenko method computes (arXiv 2106.04649; citations are /root/reference/PAPER.md
// line numbers plus SURVEY.md §8(c) step labels O1..O6).  It shares no code with the CUDA library
// (paper_2106_04649_b200/csrc) and none with the input generator.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference leg may call it.
//
// What it is: the algorithm itself, step by step, in the paper's order.  The frequency-domain shortcut
// of the paper ("performing the convolutions in the frequency domain") is replaced by
// its plain definition: a direct circular time-domain convolution (eq. 1) followed by a
// trapezoid sum over source positions, followed by the time-domain kernel of the band projector P_B.
// There is NO FFT here and no blocking / fusion / reordering beyond skipping terms that are exactly zero.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): delta-spike R => exact circular shift; linearity;
// numpy irfft(rfft*rfft) cross-check; projector idempotence / Parseval against a naive DFT; window
// support counts; the 1-D layered-medium (Goupillaud) exact case for signs, window polarity and the
// G / G+ / G- formulas; bookkeeping invariants; dense-matrix geometric series on a micro config.
// Parity unpinned (nothing in the paper fixes them; both sides use the same DESIGN.md readings):
// the absolute scale (dt, trapezoid weights), eps, the band-edge rule, the hard 0/1 window edge.
//
// Notation: n = nshot = nrec; time index j in [0,nt), negative times stored wrapped;
// (T f)[j] = f[(nt-j) % nt];  B = {klo..khi} band bins;  w[s] trapezoid weights.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

inline int wrapi(long j, int nt) {
  long m = j % nt;
  return (int)(m < 0 ? m + nt : m);
}

// (T f)[j] = f[(nt - j) % nt]   [PAPER.md:71 "iRN(t) = -iRN(-t)": the index map of t -> -t]
void time_reverse(const double* f, double* out, int nt) {
  for (int j = 0; j < nt; ++j) out[j] = f[wrapi((long)nt - j, nt)];
}

}  // namespace

extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Band B = {k in [0, nt/2] : fmin <= k df <= fmax}, df = 1/(nt dt), edges inclusive with a 1e-6-bin
// guard against rounding [DESIGN.md reading G8; "padding" implies a sub-band].  Returns nb.
int orc_band(int nt, double dt, double fmin, double fmax, int* klo, int* khi) {
  const double df = 1.0 / ((double)nt * dt);
  int lo = (int)std::ceil(fmin / df - 1e-6);
  int hi = (int)std::floor(fmax / df + 1e-6);
  lo = std::max(lo, 0);
  hi = std::min(hi, nt / 2);
  *klo = lo;
  *khi = hi;
  return hi >= lo ? hi - lo + 1 : 0;
}

// O1: trapezoid weights of the space integral of eq. (1) [PAPER.md:21 "d x"; rule: BASELINE.json north_star].
void orc_weights(int n, double dx, double* w) {
  for (int s = 0; s < n; ++s) w[s] = dx;
  if (n > 1) {
    w[0] = 0.5 * dx;
    w[n - 1] = 0.5 * dx;
  }
}

// O2: time-domain kernel of the band projector P_B (zero every DFT bin outside B, keep conjugate symmetry):
//   b[q] = (1/nt) sum_{k in B} c_k cos(2 pi k q / nt),  c_k = 1 for k in {0, nt/2}, else 2.
// A filter definition evaluated with plain cos in double — not a transform.
void orc_band_kernel(int nt, int klo, int khi, double* b) {
  const double two_pi = 6.283185307179586476925286766559;
  for (int q = 0; q < nt; ++q) {
    double acc = 0.0;
    for (int k = klo; k <= khi; ++k) {
      const double ck = (k == 0 || 2 * k == nt) ? 1.0 : 2.0;
      const long kq = ((long)k * (long)q) % nt;  // exact argument reduction
      acc += ck * std::cos(two_pi * (double)kq / (double)nt);
    }
    b[q] = acc / (double)nt;
  }
}

// y = b (*) x, circular convolution modulo nt (applies P_B to one trace).
void orc_apply_band(int nt, const double* b, const double* x, double* y) {
  for (int j = 0; j < nt; ++j) {
    double acc = 0.0;
    for (int q = 0; q < nt; ++q) acc += b[q] * x[wrapi((long)j - q, nt)];
    y[j] = acc;
  }
}

// O3: window half-width per trace, h = clamp(floor(t_d/dt + 0.5) - eps, 0, nt/2), evaluated in double
// from the fp32 traveltime; Theta[j] = 1 iff |j+-| < h  [PAPER.md:24 theta_t; readings G2, G2c].
void orc_window(int ntr, int nt, double dt, int eps, const float* td, int* h) {
  for (int i = 0; i < ntr; ++i) {
    const double m = std::floor((double)td[i] / dt + 0.5);
    double hv = m - (double)eps;
    hv = std::max(hv, 0.0);
    hv = std::min(hv, (double)(nt / 2));
    h[i] = (int)hv;
  }
}

// Theta[j] for one trace: signed index j+- = j if j < nt/2 else j - nt.
int orc_theta(int nt, int h, int j) {
  const int js = (j < nt / 2) ? j : j - nt;
  return std::abs(js) < h ? 1 : 0;
}

// O5a: synthesis without window, for a set of output receivers:
//   S[f][r][.] = P_B { dt * sum_s w[s] * sum_j' R[s][r][(j - j') % nt] * N[f][s][j'] }     [eq. (1), PAPER.md:21]
// R: [nshot][nrout][nt] fp32 (the traces of the chosen output receivers for EVERY shot),
// N: [nfoc][nshot][nt] double, S: [nfoc][nrout][nt] double.  Terms with N == 0 or R == 0 are skipped (exact).
void orc_synthesis(int nshot, int nrout, int nt, double dt, const double* w, const float* R, int nfoc,
                   const double* N, int klo, int khi, double* S) {
  std::vector<double> b(nt);
  orc_band_kernel(nt, klo, khi, b.data());

  // nonzero sample lists of N (exact skipping of zero terms)
  std::vector<std::vector<int>> nz((size_t)nfoc * nshot);
  for (int f = 0; f < nfoc; ++f)
    for (int s = 0; s < nshot; ++s) {
      const double* tr = N + ((size_t)f * nshot + s) * nt;
      auto& v = nz[(size_t)f * nshot + s];
      for (int j = 0; j < nt; ++j)
        if (tr[j] != 0.0) v.push_back(j);
    }

#pragma omp parallel
  {
    std::vector<double> acc((size_t)nfoc * 2 * nt);
    std::vector<double> Rd(nt), y(nt);
#pragma omp for schedule(dynamic, 1)
    for (int r = 0; r < nrout; ++r) {
      std::fill(acc.begin(), acc.end(), 0.0);
      for (int s = 0; s < nshot; ++s) {
        const float* Rt = R + ((size_t)s * nrout + r) * nt;
        int q0 = nt, q1 = 0;
        for (int q = 0; q < nt; ++q) {
          Rd[q] = (double)Rt[q];
          if (Rt[q] != 0.0f) {
            q0 = std::min(q0, q);
            q1 = q + 1;
          }
        }
        if (q1 <= q0) continue;
        for (int f = 0; f < nfoc; ++f) {
          const double* Nt = N + ((size_t)f * nshot + s) * nt;
          double* a = acc.data() + (size_t)f * 2 * nt;
          for (int jp : nz[(size_t)f * nshot + s]) {
            const double c = w[s] * Nt[jp];
            double* dst = a + jp;  // linear index j' + q in [0, 2nt); folded modulo nt below
            for (int q = q0; q < q1; ++q) dst[q] += c * Rd[q];
          }
        }
      }
      for (int f = 0; f < nfoc; ++f) {
        const double* a = acc.data() + (size_t)f * 2 * nt;
        for (int j = 0; j < nt; ++j) y[j] = dt * (a[j] + a[j + nt]);
        orc_apply_band(nt, b.data(), y.data(), S + ((size_t)f * nrout + r) * nt);
      }
    }
  }
}

// O4 for a set of traces (every receiver, or the chosen subset): N_{-1} = f1plus = f2 = T G_d;  f1min = pmin = 0
// [PAPER.md:19 "N_{-1} = f^+_{1,0} = G_d(-t)", 67, 74-75].  Gd: [ntr][nt] fp32; outputs [ntr][nt] double, any may be NULL.
void orc_init_subset(int ntr, int nt, const float* Gd, double* N_init, double* f1plus, double* f2, double* f1min,
                     double* pmin) {
  for (size_t i = 0; i < (size_t)ntr; ++i)
    for (int j = 0; j < nt; ++j) {
      const double v = (double)Gd[i * nt + wrapi((long)nt - j, nt)];
      if (N_init) N_init[i * nt + j] = v;
      if (f1plus) f1plus[i * nt + j] = v;
      if (f2) f2[i * nt + j] = v;
      if (f1min) f1min[i * nt + j] = 0.0;
      if (pmin) pmin[i * nt + j] = 0.0;
    }
}

// O5 for a SUBSET of output receivers (one pass of the loop body), the "single step" of
// N_prev [nfoc][nshot][nt] is the previous iterate at EVERY source position; R [nshot][nrout][nt]
// holds the traces of the chosen output receivers for every shot; h [nfoc][nrout] their window half-widths.
// Updates the subset accumulators pmin, f2, f1plus, f1min (each [nfoc][nrout][nt], any may be NULL) and writes the
// new iterate N_new [nfoc][nrout][nt] and (optionally) the unwindowed synthesis S_out.
void orc_step_subset(int nshot, int nrout, int nt, double dt, const double* w, const float* R, int nfoc,
                     const double* N_prev, const int* h, int klo, int khi, int it, double* N_new, double* S_out,
                     double* pmin, double* f2, double* f1plus, double* f1min) {
  const size_t ntr = (size_t)nfoc * nrout, tot = ntr * nt;
  std::vector<double> Sloc;
  double* S = S_out;
  if (!S) {
    Sloc.resize(tot);
    S = Sloc.data();
  }
  orc_synthesis(nshot, nrout, nt, dt, w, R, nfoc, N_prev, klo, khi, S);          // O5a [PAPER.md:69]
  if (pmin)
    for (size_t i = 0; i < tot; ++i) pmin[i] += S[i];                            // O5b [PAPER.md:79]
  for (size_t i = 0; i < ntr; ++i)                                               // O5c [PAPER.md:71-72, 78, 80]
    for (int j = 0; j < nt; ++j)
      N_new[i * nt + j] = -(double)orc_theta(nt, h[i], j) * S[i * nt + wrapi((long)nt - j, nt)];
  if (f2)
    for (size_t i = 0; i < tot; ++i) f2[i] += N_new[i];                          // O5d [PAPER.md:81]
  if (it % 2 == 0) {                                                             //     [PAPER.md:82-83]
    if (f1min)
      for (size_t i = 0; i < ntr; ++i)
        for (int j = 0; j < nt; ++j) f1min[i * nt + j] -= N_new[i * nt + wrapi((long)nt - j, nt)];
  } else {                                                                       //     [PAPER.md:84-85]
    if (f1plus)
      for (size_t i = 0; i < tot; ++i) f1plus[i] += N_new[i];
  }
}

// O6 for a SUBSET of output receivers [PAPER.md:24, 87-88; readings G3, G4, G5].  f1plus_all / f1min_all
// [nfoc][nshot][nt] are the operands of the two extra syntheses (every source position); f1plus / f1min / f2 / pmin
// [nfoc][nrout][nt] are the same fields on the chosen receivers.  Outputs [nfoc][nrout][nt], any may be NULL.
void orc_finals_subset(int nshot, int nrout, int nt, double dt, const double* w, const float* R, int nfoc,
                       const double* f1plus_all, const double* f1min_all, const double* f1plus, const double* f1min,
                       const double* f2, const double* pmin, int klo, int khi, double* G_out, double* Gplus_out,
                       double* Gminus_out) {
  const size_t ntr = (size_t)nfoc * nrout, tot = ntr * nt;
  std::vector<double> S(tot), tmp(nt);
  if (Gminus_out) {  // G- = R f1plus - f1min
    orc_synthesis(nshot, nrout, nt, dt, w, R, nfoc, f1plus_all, klo, khi, S.data());
    for (size_t i = 0; i < tot; ++i) Gminus_out[i] = S[i] - f1min[i];
  }
  if (Gplus_out) {  // G+ = T f1plus - R (T f1min)
    const size_t ntr_all = (size_t)nfoc * nshot;
    std::vector<double> Tf(ntr_all * nt);
    for (size_t i = 0; i < ntr_all; ++i) time_reverse(f1min_all + i * nt, Tf.data() + i * nt, nt);
    orc_synthesis(nshot, nrout, nt, dt, w, R, nfoc, Tf.data(), klo, khi, S.data());
    for (size_t i = 0; i < ntr; ++i) {
      time_reverse(f1plus + i * nt, tmp.data(), nt);
      for (int j = 0; j < nt; ++j) Gplus_out[i * nt + j] = tmp[j] - S[i * nt + j];
    }
  }
  if (G_out) {  // G = p- + T f2
    for (size_t i = 0; i < ntr; ++i) {
      time_reverse(f2 + i * nt, tmp.data(), nt);
      for (int j = 0; j < nt; ++j) G_out[i * nt + j] = pmin[i * nt + j] + tmp[j];
    }
  }
}

// NEXT-1: double-focusing image, the zero-time sample of G^- convolved with f1plus and integrated
// over receivers [PAPER.md:24 last sentences, 89]:  image[f] = dt sum_r w[r] sum_j G^-[f][r][(nt-j)%nt] f1plus[f][r][j].
void orc_image(int n, int nt, double dt, const double* w, int nfoc, const double* Gminus, const double* f1plus,
               double* image) {
  for (int f = 0; f < nfoc; ++f) {
    double acc = 0.0;
    for (int r = 0; r < n; ++r) {
      const double* g = Gminus + ((size_t)f * n + r) * nt;
      const double* p = f1plus + ((size_t)f * n + r) * nt;
      double part = 0.0;
      for (int j = 0; j < nt; ++j) part += g[wrapi((long)nt - j, nt)] * p[j];
      acc += w[r] * part;
    }
    image[f] = dt * acc;
  }
}

// O4..O6: the whole scheme (Algorithm 1, accumulating "on the fly" as the paper says its
// CPU version does).  Square geometry: R [n][n][nt] fp32, Gd [nfoc][n][nt] fp32, td [nfoc][n] fp32.
// Outputs (double, each [nfoc][n][nt], any may be NULL): N_iters [niter][nfoc][n][nt] (every iterate N_i),
// f1plus, f1min, f2, pmin, G, Gplus, Gminus.  Returns 0.  (The loop body and the finals are the subset routines
// above with the subset = every receiver.)
int orc_marchenko(int n, int nt, double dt, double dx, double fmin, double fmax, int eps, const float* R, int nfoc,
                  const float* Gd, const float* td, int niter, double* N_iters, double* f1plus_out,
                  double* f1min_out, double* f2_out, double* pmin_out, double* G_out, double* Gplus_out,
                  double* Gminus_out) {
  int klo, khi;
  orc_band(nt, dt, fmin, fmax, &klo, &khi);
  std::vector<double> w(n);
  orc_weights(n, dx, w.data());
  const size_t ntr = (size_t)nfoc * n, tot = ntr * nt;
  std::vector<int> h(ntr);
  orc_window((int)ntr, nt, dt, eps, td, h.data());

  // O4: N_{-1} = f1plus = f2 = T G_d;  f1min = pmin = 0      [PAPER.md:19, 67, 74-75]
  std::vector<double> N(tot), Nn(tot), f1plus(tot), f2(tot), f1min(tot), pmin(tot);
  orc_init_subset((int)ntr, nt, Gd, N.data(), f1plus.data(), f2.data(), f1min.data(), pmin.data());

  // O5: niter passes, i = 0 .. niter-1                        [PAPER.md:68, 76; reading G6]
  for (int it = 0; it < niter; ++it) {
    orc_step_subset(n, n, nt, dt, w.data(), R, nfoc, N.data(), h.data(), klo, khi, it, Nn.data(), nullptr, pmin.data(),
                    f2.data(), f1plus.data(), f1min.data());
    N.swap(Nn);
    if (N_iters) std::memcpy(N_iters + (size_t)it * tot, N.data(), tot * sizeof(double));
  }

  // O6: finals
  orc_finals_subset(n, n, nt, dt, w.data(), R, nfoc, f1plus.data(), f1min.data(), f1plus.data(), f1min.data(), f2.data(),
                    pmin.data(), klo, khi, G_out, Gplus_out, Gminus_out);
  if (f1plus_out) std::memcpy(f1plus_out, f1plus.data(), tot * sizeof(double));
  if (f1min_out) std::memcpy(f1min_out, f1min.data(), tot * sizeof(double));
  if (f2_out) std::memcpy(f2_out, f2.data(), tot * sizeof(double));
  if (pmin_out) std::memcpy(pmin_out, pmin.data(), tot * sizeof(double));
  return 0;
}

// NEXT-4: the same scheme for a spread whose sources and receivers are NOT co-located one to one.
// Eq. (1) integrates over source positions x and is evaluated at receiver positions x_R
// ("segment size is the column size (nr receivers)") keeps the two counts apart.  R [nshot][nrec][nt] fp32; G_d
// [nfoc][nrec][nt] and t_d [nfoc][nrec] live on the RECEIVER grid, and so does every output.  The operand of the next
// synthesis lives on the SHOT grid: shot s carries the trace of the receiver co-located with it, rec_of_shot[s], or
// zero when rec_of_shot[s] < 0 (no receiver there: that source position contributes nothing, the field is not known
// at it) [DESIGN.md reading G15].  w [nshot]: quadrature weights of the shot grid (irregular spacing: the caller's).
// Each iteration is orc_step_subset with "subset" = every receiver; the finals are orc_finals_subset.
int orc_marchenko_geom(int nshot, int nrec, int nt, double dt, const double* w, const int* rec_of_shot, double fmin,
                       double fmax, int eps, const float* R, int nfoc, const float* Gd, const float* td, int niter,
                       double* N_iters, double* f1plus_out, double* f1min_out, double* f2_out, double* pmin_out, double* G_out,
                       double* Gplus_out, double* Gminus_out) {
  int klo, khi;
  orc_band(nt, dt, fmin, fmax, &klo, &khi);
  const size_t ntr = (size_t)nfoc * nrec, tot = ntr * nt, tot_s = (size_t)nfoc * nshot * nt;
  std::vector<int> h(ntr);
  orc_window((int)ntr, nt, dt, eps, td, h.data());
  std::vector<double> N(tot), Nn(tot), f1plus(tot), f2(tot), f1min(tot), pmin(tot), Ns(tot_s), As(tot_s), Bs(tot_s);
  orc_init_subset((int)ntr, nt, Gd, N.data(), f1plus.data(), f2.data(), f1min.data(), pmin.data());
  // receiver grid -> shot grid: a copy of whole traces (index plumbing, no arithmetic)
  auto to_shots = [&](const std::vector<double>& src, std::vector<double>& dst) {
    for (int f = 0; f < nfoc; ++f)
      for (int s = 0; s < nshot; ++s) {
        double* d = dst.data() + ((size_t)f * nshot + s) * nt;
        const int r = rec_of_shot[s];
        if (r < 0) std::fill(d, d + nt, 0.0);
        else std::memcpy(d, src.data() + ((size_t)f * nrec + r) * nt, nt * sizeof(double));
      }
  };
  for (int it = 0; it < niter; ++it) {
    to_shots(N, Ns);
    orc_step_subset(nshot, nrec, nt, dt, w, R, nfoc, Ns.data(), h.data(), klo, khi, it, Nn.data(), nullptr, pmin.data(), f2.data(),
                    f1plus.data(), f1min.data());
    N.swap(Nn);
    if (N_iters) std::memcpy(N_iters + (size_t)it * tot, N.data(), tot * sizeof(double));
  }
  to_shots(f1plus, As);
  to_shots(f1min, Bs);
  orc_finals_subset(nshot, nrec, nt, dt, w, R, nfoc, As.data(), Bs.data(), f1plus.data(), f1min.data(), f2.data(), pmin.data(), klo,
                    khi, G_out, Gplus_out, Gminus_out);
  if (f1plus_out) std::memcpy(f1plus_out, f1plus.data(), tot * sizeof(double));
  if (f1min_out) std::memcpy(f1min_out, f1min.data(), tot * sizeof(double));
  if (f2_out) std::memcpy(f2_out, f2.data(), tot * sizeof(double));
  if (pmin_out) std::memcpy(pmin_out, pmin.data(), tot * sizeof(double));
  return 0;
}

}  // extern "C"
