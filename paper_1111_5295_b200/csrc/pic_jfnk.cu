// pic_jfnk.cu — host fp64 Jacobian-free Newton-Krylov driver (north_star (c)).
// Unknown: E^{n+1} on the faces only; the particles are enslaved state: every residual
// evaluation calls the GPU mover from state n.  Newton with a backtracking-free inexact
// Newton step; the linear solve is unpreconditioned restarted GMRES with Givens rotations and
// J w ~ [R(E + eps w) - R(E)]/eps.  Krylov residuals skip the state-(n+1) store.
#include <cmath>
#include <vector>

#include "pic_internal.h"

using namespace picb200;

namespace {

double nrm2(const std::vector<double>& a) {
  double s = 0.0;
  for (double t : a) s += t * t;
  return std::sqrt(s);
}
double dot(const std::vector<double>& a, const std::vector<double>& b) {
  double s = 0.0;
  for (size_t i = 0; i < a.size(); ++i) s += a[i] * b[i];
  return s;
}

struct Jfnk {
  pic_handle* h;    // residual handle (its state n+1 is what gets committed)
  pic_handle* hj;   // handle used for the Jacobian-vector products (== h unless defect correction)
  int n;
  int mover_calls = 0, mover_calls_j = 0;
  static int eval(pic_handle* hh, const std::vector<double>& E, std::vector<double>& R, bool store) {
    const uint32_t f0 = hh->params.flags;
    hh->params.flags = store ? (f0 & ~PIC_FLAG_NO_STORE) : (f0 | PIC_FLAG_NO_STORE);
    const bool keep = hh->have_np1;
    const int rc = residual_impl(hh, E.data(), R.data(), 0, 0);   // host vectors
    if (!store) hh->have_np1 = keep;   // a Krylov call leaves the stored state n+1 untouched
    hh->params.flags = f0;
    return rc;
  }
  // true residual (stores state n+1)
  int resid(const std::vector<double>& E, std::vector<double>& R) {
    ++mover_calls;
    return eval(h, E, R, true);
  }
  // residual as the Jacobian handle sees it (no store)
  int resid_j(const std::vector<double>& E, std::vector<double>& R) {
    ++mover_calls_j;
    return eval(hj, E, R, false);
  }
};

int jfnk_core(pic_handle* h, pic_handle* hj, double* E, double dt, double tol,
              const pic_jfnk_opts* opts, pic_jfnk_info* info);

}  // namespace

namespace {
int jfnk_core(pic_handle* h, pic_handle* hj, double* E, double dt, double tol,
              const pic_jfnk_opts* opts, pic_jfnk_info* info) {
  if (!h || !hj) return PIC_ERR_ARG;
  if (!E || !(dt > 0.0)) return set_err(h, PIC_ERR_ARG, "pic_jfnk_step: bad argument");
  if (is_device_ptr(E)) return set_err(h, PIC_ERR_ARG, "pic_jfnk_step: E must be a host array");
  pic_jfnk_opts o;
  if (opts) o = *opts;
  else o = pic_jfnk_opts{1e-8, 0.0, 0.0, 1e-2, 20, 30, 200, 0};
  if (o.fd_eps <= 0.0) o.fd_eps = hj->elem == 4 ? 1e-3 : 1e-6;
  if (o.max_newton < 1) o.max_newton = 20;
  if (o.gmres_restart < 1) o.gmres_restart = 30;
  if (o.max_gmres < 1) o.max_gmres = 200;
  if (o.gmres_rtol <= 0.0) o.gmres_rtol = 1e-2;
  const int n = h->grid.n_cells;
  int rc = pic_set_step(h, E, dt, tol);
  if (rc != PIC_OK) return rc;
  const bool dc = hj != h;   // defect correction: J w from the other (fp32) mover
  if (dc) {
    if (hj->grid.n_cells != n || hj->sp.size() != h->sp.size())
      return set_err(h, PIC_ERR_ARG, "pic_jfnk_step_dc: the two handles differ in grid or species");
    if ((rc = pic_set_step(hj, E, dt, tol)) != PIC_OK) return rc;
  }
  Jfnk J{h, hj, n};
  std::vector<double> Rj0(n);   // residual of the Jacobian handle at the Newton iterate
  std::vector<double> Ek(E, E + n), R(n), Rp(n), w(n), Ep(n);
  if ((rc = J.resid(Ek, R)) != PIC_OK && rc != PIC_ERR_SUBSTEP_CAP) return rc;
  bool capped = rc == PIC_ERR_SUBSTEP_CAP;   // of the LAST true residual (the state to commit)
  const double r0 = nrm2(R);
  double rn = r0;
  int newton = 0, gm_total = 0;
  bool conv = rn <= o.atol;
  const int m = o.gmres_restart;
  std::vector<std::vector<double>> V(m + 1, std::vector<double>(n));
  std::vector<double> Hm((size_t)(m + 1) * m), cs(m), sn(m), g(m + 1), y(m), dE(n);
  while (!conv && newton < o.max_newton) {
    // ---- GMRES(m) on J dE = -R, dE_0 = 0
    // base point of the finite differences: with defect correction the Jacobian handle's own
    // residual at E_k (one extra fp32 call per Newton step), else R itself
    if (dc) {
      if ((rc = J.resid_j(Ek, Rj0)) != PIC_OK && rc != PIC_ERR_SUBSTEP_CAP) return rc;
    } else {
      Rj0 = R;
    }
    std::fill(dE.begin(), dE.end(), 0.0);
    const double En = nrm2(Ek);
    const double lin_tol = o.gmres_rtol * rn;
    int gm_it = 0;
    double lin_res = rn;
    std::vector<double> rhs(n);
    for (int i = 0; i < n; ++i) rhs[i] = -R[i];
    bool lin_done = false;
    while (!lin_done && gm_it < o.max_gmres) {
      // residual of the linear system: rhs - J dE  (first cycle: dE = 0)
      std::vector<double>& v0 = V[0];
      if (gm_it == 0) v0 = rhs;
      else {
        const double dn = nrm2(dE);
        const double eps = o.fd_eps * (1.0 + En) / (dn > 0 ? dn : 1.0);
        for (int i = 0; i < n; ++i) Ep[i] = Ek[i] + eps * dE[i];
        if ((rc = J.resid_j(Ep, Rp)) != PIC_OK && rc != PIC_ERR_SUBSTEP_CAP) return rc;
        for (int i = 0; i < n; ++i) v0[i] = rhs[i] - (Rp[i] - Rj0[i]) / eps;
      }
      double beta = nrm2(v0);
      if (beta <= lin_tol) { lin_res = beta; break; }
      for (int i = 0; i < n; ++i) v0[i] /= beta;
      std::fill(g.begin(), g.end(), 0.0);
      g[0] = beta;
      int k = 0;
      for (; k < m && gm_it < o.max_gmres; ++k, ++gm_it) {
        const double eps = o.fd_eps * (1.0 + En);   // ||V[k]|| = 1
        for (int i = 0; i < n; ++i) Ep[i] = Ek[i] + eps * V[k][i];
        if ((rc = J.resid_j(Ep, Rp)) != PIC_OK && rc != PIC_ERR_SUBSTEP_CAP) return rc;
        for (int i = 0; i < n; ++i) w[i] = (Rp[i] - Rj0[i]) / eps;
        for (int j = 0; j <= k; ++j) {   // modified Gram-Schmidt
          const double hjk = dot(w, V[j]);
          Hm[(size_t)j * m + k] = hjk;
          for (int i = 0; i < n; ++i) w[i] -= hjk * V[j][i];
        }
        const double hk1 = nrm2(w);
        Hm[(size_t)(k + 1) * m + k] = hk1;
        if (hk1 > 0) for (int i = 0; i < n; ++i) V[k + 1][i] = w[i] / hk1;
        for (int j = 0; j < k; ++j) {   // apply earlier rotations
          const double t = cs[j] * Hm[(size_t)j * m + k] + sn[j] * Hm[(size_t)(j + 1) * m + k];
          Hm[(size_t)(j + 1) * m + k] = -sn[j] * Hm[(size_t)j * m + k] + cs[j] * Hm[(size_t)(j + 1) * m + k];
          Hm[(size_t)j * m + k] = t;
        }
        const double a = Hm[(size_t)k * m + k], b = Hm[(size_t)(k + 1) * m + k];
        const double rr = std::hypot(a, b);
        cs[k] = rr > 0 ? a / rr : 1.0;
        sn[k] = rr > 0 ? b / rr : 0.0;
        Hm[(size_t)k * m + k] = rr;
        Hm[(size_t)(k + 1) * m + k] = 0.0;
        g[k + 1] = -sn[k] * g[k];
        g[k] = cs[k] * g[k];
        lin_res = std::fabs(g[k + 1]);
        if (lin_res <= lin_tol || hk1 == 0.0) { ++k; ++gm_it; lin_done = true; break; }
      }
      for (int i = k - 1; i >= 0; --i) {   // back substitution
        double s = g[i];
        for (int j = i + 1; j < k; ++j) s -= Hm[(size_t)i * m + j] * y[j];
        y[i] = s / Hm[(size_t)i * m + i];
      }
      for (int j = 0; j < k; ++j)
        for (int i = 0; i < n; ++i) dE[i] += y[j] * V[j][i];
    }
    gm_total += gm_it;
    // ---- Newton update and new residual (stores state n+1)
    for (int i = 0; i < n; ++i) Ek[i] += dE[i];
    if ((rc = J.resid(Ek, R)) != PIC_OK && rc != PIC_ERR_SUBSTEP_CAP) return rc;
    capped = rc == PIC_ERR_SUBSTEP_CAP;
    rn = nrm2(R);
    ++newton;
    conv = rn <= o.rtol * r0 || rn <= o.atol;
  }
  if (info) {
    info->newton_its = newton;
    info->gmres_its = gm_total;
    info->mover_calls = J.mover_calls + J.mover_calls_j;
    info->mover_calls_resid = J.mover_calls;
    info->converged = conv ? 1 : 0;
    info->resid0 = r0;
    info->resid = rn;
  }
  // A rejected step leaves the caller where it was: E still holds E^n and the particles are at
  // state n, so the step can be retried (smaller dt, larger max_substeps); E^{n+1} is delivered
  // only together with the committed particle state.
  if (!conv)
    return set_err(h, PIC_ERR_STATE,
                   "pic_jfnk_step: Newton did not converge (E left at E^n, state not committed)");
  if (capped)   // A-9: some orbits of the converged state did not use up dt
    return set_err(h, PIC_ERR_SUBSTEP_CAP,
                   "pic_jfnk_step: particles cut off at max_substeps (E left at E^n, state not committed)");
  if ((rc = pic_commit(h)) != PIC_OK) return rc;
  for (int i = 0; i < n; ++i) E[i] = Ek[i];
  if (dc) return pic_copy_state(hj, h);   // the Jacobian handle follows the committed state
  return PIC_OK;
}
}  // namespace

extern "C" int pic_jfnk_step(pic_handle* h, double* E, double dt, double tol,
                             const pic_jfnk_opts* opts, pic_jfnk_info* info) {
  return jfnk_core(h, h, E, dt, tol, opts, info);
}

extern "C" int pic_jfnk_step_dc(pic_handle* h_resid, pic_handle* h_jac, double* E, double dt,
                                double tol, const pic_jfnk_opts* opts, pic_jfnk_info* info) {
  if (h_resid == h_jac) return h_resid ? set_err(h_resid, PIC_ERR_ARG, "pic_jfnk_step_dc: need two handles") : PIC_ERR_ARG;
  return jfnk_core(h_resid, h_jac, E, dt, tol, opts, info);
}
