// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, serial, double-precision restatement of the implicit, adaptive,
// charge-conserving particle mover of Chen, Chacon & Barnes (arXiv 1111.5295),
// written from /root/reference/PAPER.md ("P:<line>") with the readings listed in
// SURVEY.md section 8(c) (O1..O11, A-1..A-17) and DESIGN.md section 3.
//
// It shares NO code with the CUDA path (paper_1111_5295_b200/csrc) and is imported
// only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs.  It follows the paper's order of operations, one particle at
// a time, one sub-step at a time; there is no blocking, fusion or reordering.
//
// Pins (tests/test_oracle_pins.py): P-1 free streaming, P-2 uniform field parabola,
// P-3 Eq. 11 == Picard fixed point, P-4 estimator bound, P-5 crossing invariants +
// bisection, P-6 per-cell discrete continuity, P-7 endpoint formula, P-8 mean current,
// P-9 energy identity, P-10 refinement to the harmonic oscillator / RK reference,
// P-11 hand-stepped tiny cases, P-12 residual sum; the A-9 sub-step cap (prefix property of the
// aborted orbit); oracle_bin against hand values and the
// identity cell*dx + s = x; and pins on workloads that EXECUTE the guard branches: the A-2
// kappa cap (binding on most sub-steps), the O7 discriminant and crossing-time clamps
// (rounding coincidences: particles that end a step exactly on a face), the A-3 Picard cap
// (picard_max = 1 is the explicit midpoint rule) -- each checked against what the mathematics
// still fixes there (1 - kappa >= 1/2, sum dtau = dt, closed-form end state, P-5, P-6, P-9).
// Every function of this file is pinned and every branch is executed by a pin (gcov: 294 of 300
// lines under tests/test_oracle_pins.py), except three defensive guards that no input can reach
// (DESIGN.md section 2): `dtau_c = dtau` for a_m == 0 while moving away from the exit face, the
// lower clamp `dtau_c = 0` (a negative or NaN crossing time), and `w = 0` beyond the support of
// the quadratic spline in oracle_rho (|xi| <= 3/2 always holds for the three cells visited).
// What no pin can
// settle is where the PAPER is silent and a reading had to be chosen:
// the value kappa_max = 0.5 (A-2), the form of the Picard convergence test (A-3), the face
// convention (A-5), the sub-step cap (A-9), the face/cell index convention.  The code that
// implements each reading is pinned as above; the choice itself is a reading, not a result.
//
// Conventions (SURVEY 8 "Common notation"): periodic [0,L), n_cells uniform cells,
// dx = L/n_cells; face f at x_f = f*dx; cell c spans faces c and (c+1) mod n_cells.
// E and the current live on faces; rho lives on cell centres.
// Particle state: cell index c (authoritative, P:123 carries i_p), in-cell offset
// s = x - x_c in [0,dx], velocity v.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

struct oracle_params {
  double eps_a;         // absolute tolerance of the sub-step estimator (1e-8)
  double eps_r;         // relative tolerance (0.02)
  double kappa_max;     // A-2 cap on |a' dtau^2/4| (0.5)
  double tol;           // Picard tolerance (A-3)
  int32_t max_substeps; // A-9 cap (2^20)
  int32_t cn_mode;      // 0 = Picard iteration of Eq. 9-10, 1 = direct Eq. 11
  int32_t picard_max;   // iteration cap of the Picard loop (100)
  int32_t pad_;
};

struct oracle_stats {
  int64_t n_sub;         // total sub-steps
  int64_t n_cross;       // total cell crossings
  int64_t n_picard_it;   // total Picard iterations
  int64_t n_picard_cap;  // sub-steps whose Picard loop hit picard_max
  int64_t n_kappa_cap;   // sub-steps whose dtau was limited by the A-2 cap
  int64_t n_substep_cap; // particles aborted at max_substeps
  int64_t n_neg_disc;    // crossings whose discriminant v^2+2 a_m d was clamped at 0
  int64_t n_clamped_tau; // crossings whose dtau_c was clamped to [0,dtau]
};

// One record per sub-step, for the tests that look inside an orbit (P-4, P-5, P-11).
struct oracle_substep {
  double dtau_est;  // estimator output before min(.,r) and the kappa cap
  double dtau;      // sub-step actually taken
  double s0, v0;    // state at the start of the sub-step
  double s1, v1;    // state at its end
  double a, aprime; // a(s0) and a' of the cell
  double a_mid;     // acceleration used by the step (midpoint value)
  int32_t cell;     // cell during the sub-step
  int32_t crossed;  // 0 in-cell, +1 left through the right face, -1 through the left face
};

}  // extern "C"

namespace {

struct Trace {
  oracle_substep* rec;
  int64_t cap;
  int64_t n;
};

// O4 — sub-step estimator, Eq. 6-8 in its L1 / max form:
//   alpha = (|a| + |a' v|)/2, beta = eps_r (|a| + |v|), gamma^2 = eps_a,
//   dtau = max(gamma d, beta d^2), d = alpha^(-1/2).
// A-1: alpha is floored at the smallest normal so that E = 0 gives dtau = huge -> r.
inline double estimate_dtau(double a, double aprime, double v, double eps_a, double eps_r) {
  double alpha = 0.5 * (std::fabs(a) + std::fabs(aprime * v));
  if (alpha < 1e-300) alpha = 1e-300;
  const double beta = eps_r * (std::fabs(a) + std::fabs(v));
  const double t_abs = std::sqrt(eps_a / alpha);  // Eq. 7
  const double t_rel = beta / alpha;              // Eq. 8
  return t_abs > t_rel ? t_abs : t_rel;
}

}  // namespace

namespace {

// O2-O9 for one particle.  J (length n_cells, raw: sum of w_q*delta*weight, not yet
// divided by dt*dx) is accumulated in place.  Returns the number of sub-steps.
void move_one(int n_cells, double dx, double q_over_m, double w_q, const double* Ehalf,
              const oracle_params& p, double dt, int32_t& c, double& s, double& v, int32_t& k,
              uint32_t& n_sub, uint32_t& n_cross, double* J, oracle_stats& st, Trace* tr) {
  double r = dt;  // O2: remaining time
  n_sub = 0;
  n_cross = 0;
  k = 0;
  while (r > 0.0) {
    if ((int64_t)n_sub >= (int64_t)p.max_substeps) {  // A-9
      st.n_substep_cap++;
      break;
    }
    // O3 — cell constants (Eq. 5): a' = (q/m)(E_{c+1}-E_c)/dx, a = a_L + a' s.
    const int cr = (c + 1) % n_cells;
    const double a_L = q_over_m * Ehalf[c];
    const double a_R = q_over_m * Ehalf[cr];
    const double aprime = (a_R - a_L) / dx;
    const double a = a_L + aprime * s;

    // O4 — estimator, then dtau = min(dtau_est, kappa cap, r).
    const double dtau_est = estimate_dtau(a, aprime, v, p.eps_a, p.eps_r);
    double dtau = dtau_est;
    if (aprime != 0.0) {  // A-2: |kappa| = |a'| dtau^2/4 <= kappa_max
      const double cap = std::sqrt(4.0 * p.kappa_max / std::fabs(aprime));
      if (dtau > cap) {
        dtau = cap;
        st.n_kappa_cap++;
      }
    }
    if (dtau > r) dtau = r;

    // O5 — tentative Crank-Nicolson step over dtau (Eq. 9-10), using the
    // linear field of the CURRENT cell even if the midpoint leaves it (A-4).
    double v1, a_mid;
    if (p.cn_mode == 0) {
      // Picard: v' <- v; iterate v'' = v + dtau * a(s + dtau (v+v')/4).
      double vk = v;
      int it = 0;
      for (;;) {
        const double s_m = s + dtau * (v + vk) / 4.0;
        a_mid = a_L + aprime * s_m;
        const double vn = v + dtau * a_mid;
        ++it;
        const bool done = std::fabs(vn - vk) <= p.tol * (std::fabs(vn) + std::fabs(a_mid) * dtau);
        vk = vn;
        if (done) break;
        if (it >= p.picard_max) {
          st.n_picard_cap++;
          break;
        }
      }
      st.n_picard_it += it;
      v1 = vk;
    } else {
      // Direct solve, Eq. 11: kappa = a' dtau^2/4,
      //   v' = [a dtau + (1+kappa) v] / (1-kappa).
      const double kappa = aprime * dtau * dtau / 4.0;
      v1 = (a * dtau + (1.0 + kappa) * v) / (1.0 - kappa);
      a_mid = a_L + aprime * (s + dtau * (v + v1) / 4.0);
    }
    const double s1 = s + dtau * (v + v1) / 2.0;  // Eq. 9

    oracle_substep rec;
    rec.dtau_est = dtau_est;
    rec.s0 = s;
    rec.v0 = v;
    rec.a = a;
    rec.aprime = aprime;
    rec.cell = c;

    if (s1 >= 0.0 && s1 <= dx) {
      // O6 — accept (inclusive test, A-5).  O8 deposit with delta = s1 - s.
      const double delta = s1 - s;
      const double w_R = (s + s1) / (2.0 * dx);
      J[cr] += w_q * delta * w_R;
      J[c] += w_q * delta * (1.0 - w_R);
      rec.dtau = dtau;
      rec.s1 = s1;
      rec.v1 = v1;
      rec.a_mid = a_mid;
      rec.crossed = 0;
      s = s1;
      v = v1;
      r = (dtau == r) ? 0.0 : r - dtau;
      n_sub++;
    } else {
      // O7 — crossing: land on the face the tentative step left through.
      const int sigma = (s1 > dx) ? +1 : -1;
      const double d = (sigma > 0) ? (dx - s) : (-s);  // signed distance to that face
      const double a_m = a + aprime * d / 2.0;         // a at the midpoint of the truncated step
      double D = v * v + 2.0 * a_m * d;                // Eq. 12 (energy principle)
      if (D < 0.0) {
        D = 0.0;
        st.n_neg_disc++;
      }
      const double vc = sigma * std::sqrt(D);
      // Root of F(dtau) = (a_m/2) dtau^2 + v dtau - d.  A-6: Eq. 13 as printed is
      // (vc - v)/a_m; when the particle already moves towards the face use the
      // algebraically identical 2d/(v+vc), which has no cancellation and no 0/0.
      double dtau_c;
      if (sigma * v > 0.0)
        dtau_c = 2.0 * d / (v + vc);
      else if (a_m != 0.0)
        dtau_c = (vc - v) / a_m;
      else
        dtau_c = dtau;
      if (!(dtau_c >= 0.0)) {
        dtau_c = 0.0;
        st.n_clamped_tau++;
      } else if (dtau_c > dtau) {
        dtau_c = dtau;
        st.n_clamped_tau++;
      }
      // O8 deposit with delta = d; the end point is the face exactly.
      const double s_end = (sigma > 0) ? dx : 0.0;
      const double w_R = (s + s_end) / (2.0 * dx);
      J[cr] += w_q * d * w_R;
      J[c] += w_q * d * (1.0 - w_R);
      rec.dtau = dtau_c;
      rec.s1 = s_end;
      rec.v1 = vc;
      rec.a_mid = a_m;
      rec.crossed = sigma;
      // enter the neighbouring cell on its near face
      s = (sigma > 0) ? 0.0 : dx;
      c = (sigma > 0) ? cr : (c + n_cells - 1) % n_cells;
      k += sigma;
      v = vc;
      r = (dtau_c == r) ? 0.0 : r - dtau_c;
      n_sub++;
      n_cross++;
    }
    if (tr && tr->n < tr->cap) tr->rec[tr->n++] = rec;
  }
}

}  // namespace

extern "C" {

// Position -> (cell, offset).  cell = floor(x/dx) clipped to [0, n_cells-1]; s = x - cell*dx
// clipped to [0, dx].
void oracle_bin(int32_t n_cells, double length, int64_t n, const double* x, int32_t* cell,
                double* s) {
  const double dx = length / n_cells;
  for (int64_t p = 0; p < n; ++p) {
    int32_t c = (int32_t)std::floor(x[p] / dx);
    if (c < 0) c = 0;
    if (c > n_cells - 1) c = n_cells - 1;
    double sp = x[p] - c * dx;
    if (sp < 0.0) sp = 0.0;
    if (sp > dx) sp = dx;
    cell[p] = c;
    s[p] = sp;
  }
}

// O1-O9 for one species.  Inputs: state n as (cell0, s0, v0); E_n, E_np1 on faces.
// Outputs (any may be NULL): state n+1 (cell1, s1, v1), k_net = signed net number of cells
// crossed, per-particle n_sub / n_cross.  J [n_cells] is ACCUMULATED (raw, un-normalised) so
// that several species can be summed by calling this once per species; stats likewise.
int oracle_move_accumulate(int32_t n_cells, double length, double q_over_m, double w_q,
                           int64_t n, const int32_t* cell0, const double* s0, const double* v0,
                           const double* E_n, const double* E_np1, double dt,
                           const oracle_params* params, int32_t* cell1, double* s1, double* v1,
                           int32_t* k_net, uint32_t* n_sub, uint32_t* n_cross, double* J,
                           oracle_stats* stats) {
  if (n_cells < 1 || !(length > 0.0) || !(dt >= 0.0) || !params || !J || !stats) return -1;
  const double dx = length / n_cells;
  // O1 — E^{n+1/2} = (E^n + E^{n+1})/2 on faces (BASELINE.json north_star; A-11).
  std::vector<double> Ehalf(n_cells);
  for (int f = 0; f < n_cells; ++f) Ehalf[f] = 0.5 * (E_n[f] + E_np1[f]);
  for (int64_t p = 0; p < n; ++p) {
    int32_t c = cell0[p];
    double s = s0[p], v = v0[p];
    if (c < 0 || c >= n_cells || !(s >= 0.0 && s <= dx) || !std::isfinite(v)) return -2;
    int32_t k;
    uint32_t ns, nc;
    move_one(n_cells, dx, q_over_m, w_q, Ehalf.data(), *params, dt, c, s, v, k, ns, nc, J,
             *stats, nullptr);
    stats->n_sub += ns;
    stats->n_cross += nc;
    if (cell1) cell1[p] = c;
    if (s1) s1[p] = s;
    if (v1) v1[p] = v;
    if (k_net) k_net[p] = k;
    if (n_sub) n_sub[p] = ns;
    if (n_cross) n_cross[p] = nc;
  }
  return 0;
}

// Same mover for ONE particle, recording every sub-step.  Returns the number of records
// written (<= cap), or a negative error.
int64_t oracle_trace_particle(int32_t n_cells, double length, double q_over_m, double w_q,
                              int32_t cell0, double s0, double v0, const double* E_n,
                              const double* E_np1, double dt, const oracle_params* params,
                              oracle_substep* rec, int64_t cap, int32_t* cell1, double* s1,
                              double* v1, int32_t* k_net, double* J) {
  if (n_cells < 1 || !(length > 0.0) || !params || !J) return -1;
  const double dx = length / n_cells;
  std::vector<double> Ehalf(n_cells);
  for (int f = 0; f < n_cells; ++f) Ehalf[f] = 0.5 * (E_n[f] + E_np1[f]);
  oracle_stats st;
  std::memset(&st, 0, sizeof st);
  Trace tr{rec, cap, 0};
  int32_t c = cell0, k;
  double s = s0, v = v0;
  uint32_t ns, nc;
  move_one(n_cells, dx, q_over_m, w_q, Ehalf.data(), *params, dt, c, s, v, k, ns, nc, J, st, &tr);
  if (cell1) *cell1 = c;
  if (s1) *s1 = s;
  if (v1) *v1 = v;
  if (k_net) *k_net = k;
  return tr.n;
}

// Stand-alone estimator (for pin P-4).
double oracle_estimate_dtau(double a, double aprime, double v, double eps_a, double eps_r) {
  return estimate_dtau(a, aprime, v, eps_a, eps_r);
}

// O10 — orbit average: jbar_f = J_f / (dt * dx).
void oracle_jbar(int32_t n_cells, double length, double dt, const double* J, double* jbar) {
  const double dx = length / n_cells;
  for (int f = 0; f < n_cells; ++f) jbar[f] = J[f] / (dt * dx);
}

// a9 — Ampere residual (north_star): R_f = eps0 (E^{n+1}_f - E^n_f)/dt + jbar_f - <jbar>,
// <jbar> = (1/n_cells) sum_f jbar_f, eps0 = 1.
void oracle_residual(int32_t n_cells, const double* E_n, const double* E_np1, double dt,
                     const double* jbar, double* resid) {
  double mean = 0.0;
  for (int f = 0; f < n_cells; ++f) mean += jbar[f];
  mean /= n_cells;
  for (int f = 0; f < n_cells; ++f) resid[f] = (E_np1[f] - E_n[f]) / dt + jbar[f] - mean;
}

// O11 — charge density on cell centres with the quadratic B-spline (A-10):
//   rho_c += (w_q/dx) * S2((x_centre,c - x_p)/dx),
//   S2(xi) = 3/4 - xi^2 (|xi| <= 1/2), (3/2 - |xi|)^2 / 2 (1/2 <= |xi| <= 3/2), else 0.
// rho [n_cells] is ACCUMULATED (several species).
void oracle_rho(int32_t n_cells, double length, double w_q, int64_t n, const int32_t* cell,
                const double* s, double* rho) {
  const double dx = length / n_cells;
  for (int64_t p = 0; p < n; ++p) {
    const int c = cell[p];
    const double u = s[p] / dx;  // position in the cell, 0..1
    for (int m = -1; m <= 1; ++m) {
      const double xi = std::fabs((m + 0.5) - u);  // distance to the centre of cell c+m
      double w;
      if (xi <= 0.5)
        w = 0.75 - xi * xi;
      else if (xi <= 1.5)
        w = 0.5 * (1.5 - xi) * (1.5 - xi);
      else
        w = 0.0;
      rho[((c + m) % n_cells + n_cells) % n_cells] += w_q * w / dx;
    }
  }
}

}  // extern "C"
