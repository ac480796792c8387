// mover.cuh — the implicit, adaptive, charge-conserving particle mover kernel (sm_100a).
//
// One launch = steps a0..a8 of SURVEY.md 8(a) for one species: field prologue,
// per-particle sub-step loop {estimate dtau (Eq. 6-8) -> Crank-Nicolson move
// (Eq. 9-11) -> cell-crossing truncation (Eq. 12-14)}, current deposit
// into per-block shared-memory accumulators, one flush per block.
//
// Shares no code with oracle/.  Design notes:
//  * all per-particle arithmetic is in CELL UNITS: xi = (x - x_c)/dx in [0,1], u = v/dx,
//    A_f = (q/m) E^{n+1/2}_f / dx.  Inside cell c: A(xi) = A_L + dA xi, dA = A_R - A_L = a'.
//  * the deposit uses the telescoped per-cell-visit form of the per-sub-step sum (SURVEY P-7):
//    a stay in one cell from xi_in to xi_out contributes delta*m to the right face and
//    delta*(1-m) to the left face, delta = xi_out - xi_in, m = (xi_in + xi_out)/2 -- the sum of
//    P:212's per-sub-step linear-spline deposits over that stay, to rounding.  It is flushed to
//    shared memory on crossing / at orbit end (the paper's register accumulation).
//  * divergence (variable sub-step counts): persistent warps; a lane whose
//    orbit is finished parks its result and, once enough lanes of the warp are parked, the
//    parked lanes store and pull the next particles of the warp's current index range
//    (lane-level re-queue); ranges are claimed from a global counter.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace picb200 {

constexpr int kBlock = 512;        // threads per block
constexpr unsigned kFull = 0xffffffffu;

enum StatSlot { ST_SUB = 0, ST_CROSS, ST_PICARD_IT, ST_PICARD_CAP, ST_KAPPA_CAP, ST_SUBSTEP_CAP,
                ST_NEG_DISC, ST_CLAMPED, ST_COUNT };

template <typename T>
struct MoverArgs {
  long long n;                 // particles of this species
  const T* xi0;                // state n, SoA, binned by cell
  const T* v0;
  const int32_t* cell0;
  T* xi1;                      // state n+1 (same order); may be NULL (PIC_FLAG_NO_STORE)
  T* v1;
  int32_t* cell1;
  uint32_t* nsub_out;          // optional per-particle counts (PIC_FLAG_COUNTS)
  uint32_t* ncross_out;
  const double* E_n;           // faces, device
  const double* E_np1;
  int32_t n_cells;
  int32_t max_substeps;
  int32_t picard_max;
  int32_t tile;                // particles per claimed index range (multiple of 32)
  int32_t refill_threshold;    // parked lanes needed before a refill
  double qm_over_dx;           // (q/m)/dx
  T dx, inv_dx;
  T c_abs;                     // sqrt(2 eps_a / dx):   dtau_abs = c_abs / sqrt(|A| + |dA u|)
  T c_rel;                     // 2 eps_r:              dtau_rel = c_rel (|A|+|u|) / (|A|+|dA u|)
  T c_cap;                     // sqrt(4 kappa_max):    dtau_cap = c_cap / sqrt(|dA|)
  T dt, tol;
  double scale;                // w_q / dt : cell-unit deposit -> jbar contribution
  double* partial;             // [gridDim.x][n_cells] per-block sums (scaled)
  unsigned long long* queue;   // global index-range counter (zeroed before launch)
  unsigned long long* stats;   // [ST_COUNT] totals (accumulated)
};

// ---- precision-specific primitives -------------------------------------------------------
template <typename T> struct Prim;

template <> struct Prim<float> {
  static __device__ __forceinline__ float rsqrt(float x) {  // MUFU.RSQ
    float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float rcp(float x) {    // MUFU.RCP
    float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float sqrt(float x) {   // MUFU.SQRT
    float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float div(float a, float b) { return a * rcp(b); }
  static __device__ __forceinline__ float tiny() { return 1e-30f; }
  static __device__ __forceinline__ float eps() { return 1.1920929e-7f; }
};

template <> struct Prim<double> {
  static __device__ __forceinline__ double rsqrt(double x) { return 1.0 / ::sqrt(x); }
  static __device__ __forceinline__ double rcp(double x) { return 1.0 / x; }
  static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
  static __device__ __forceinline__ double div(double a, double b) { return a / b; }
  static __device__ __forceinline__ double tiny() { return 1e-300; }
  static __device__ __forceinline__ double eps() { return 2.220446049250313e-16; }
};

template <typename T> __device__ __forceinline__ T tabs(T x);
template <> __device__ __forceinline__ float tabs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double tabs<double>(double x) { return fabs(x); }
template <typename T> __device__ __forceinline__ T tmin(T a, T b) { return a < b ? a : b; }
template <typename T> __device__ __forceinline__ T tmax(T a, T b) { return a > b ? a : b; }
template <> __device__ __forceinline__ float tmin<float>(float a, float b) { return fminf(a, b); }
template <> __device__ __forceinline__ float tmax<float>(float a, float b) { return fmaxf(a, b); }
template <> __device__ __forceinline__ double tmin<double>(double a, double b) { return fmin(a, b); }
template <> __device__ __forceinline__ double tmax<double>(double a, double b) { return fmax(a, b); }

// Per-lane particle registers.
template <typename T>
struct Lane {
  T xi, u, r;          // in-cell offset, velocity in cells/time, remaining time (O2)
  T AL, dA, cap;       // constants of the current cell (O3) and its kappa cap (A-2)
  T xin;               // xi at entry into the current cell (telescoped deposit)
  int32_t c;           // cell
  uint32_t ns, nc;     // sub-steps, crossings of this orbit
  long long idx;       // particle index; -1 = nothing parked
};

// O3: constants of cell c from the staged face values.
template <typename T>
__device__ __forceinline__ void load_cell(const T* __restrict__ sA, int32_t n_cells, T c_cap,
                                          Lane<T>& p) {
  const int32_t cr = (p.c + 1 == n_cells) ? 0 : p.c + 1;
  const T AL = sA[p.c], AR = sA[cr];
  p.AL = AL;
  p.dA = AR - AL;
  // A-2: dtau <= sqrt(4 kappa_max / |a'|); |dA| = 0 gives +inf (no cap).
  p.cap = c_cap * Prim<T>::rsqrt(tabs(p.dA));
}

// a5/O8 (telescoped): flush the stay [xin, xout] in cell c to the block accumulators.
template <typename T>
__device__ __forceinline__ void deposit(double* __restrict__ sJ, int32_t n_cells, int32_t c,
                                        T xin, T xout) {
  const T delta = xout - xin;
  const T right = delta * (T(0.5) * (xin + xout));
  const T left = delta - right;
  const int32_t cr = (c + 1 == n_cells) ? 0 : c + 1;
  atomicAdd(&sJ[c], (double)left);
  atomicAdd(&sJ[cr], (double)right);
}

// One sub-step (O3-O8) of the lane's particle.  CN_DIRECT: Eq. 11, else Picard on Eq. 9-10.
template <typename T, bool CN_DIRECT, bool DIAG>
__device__ __forceinline__ void substep(const MoverArgs<T>& a, const T* __restrict__ sA,
                                        double* __restrict__ sJ, Lane<T>& p,
                                        unsigned& picard_its, unsigned* diag) {
  // ---- a2 / O4: estimator (Eq. 6-8), L1 form, in cell units:
  //   alpha = dx (|A| + |dA u|)/2, beta = eps_r dx (|A| + |u|)
  //   dtau = max( sqrt(eps_a/alpha), beta/alpha ) = max( c_abs d, c_rel (|A|+|u|) d^2 ),
  //   d = (|A| + |dA u|)^(-1/2)  (one rsqrt).  A-1: floor the sum at `tiny`.
  const T A = fma(p.dA, p.xi, p.AL);
  const T absA = tabs(A);
  const T S = tmax(absA + tabs(p.dA * p.u), Prim<T>::tiny());
  const T d = Prim<T>::rsqrt(S);
  T dtau = tmax(a.c_abs * d, (a.c_rel * (absA + tabs(p.u))) * (d * d));
  if (DIAG && dtau > p.cap) diag[ST_KAPPA_CAP]++;
  dtau = tmin(tmin(dtau, p.cap), p.r);

  // ---- a3 / O5: tentative Crank-Nicolson step over dtau with the linear field of the
  // current cell (A-4).
  T u1;
  if (CN_DIRECT) {
    // Eq. 11: kappa = a' dtau^2/4;  u' = [A dtau + (1+kappa) u] / (1-kappa).
    const T kappa = (T(0.25) * p.dA) * (dtau * dtau);
    const T num = fma(A, dtau, fma(kappa, p.u, p.u));
    u1 = Prim<T>::div(num, T(1) - kappa);
  } else {
    // Picard (A-3): u' <- u; u'' = u + dtau A(xi + dtau (u+u')/4) until
    // |u''-u'| <= tol (|u''| + |A_m| dtau).
    T uk = p.u;
    int it = 0;
    for (;;) {
      const T xim = fma(T(0.25) * dtau, p.u + uk, p.xi);
      const T Am = fma(p.dA, xim, p.AL);
      const T un = fma(dtau, Am, p.u);
      ++it;
      const bool done = tabs(un - uk) <= a.tol * (tabs(un) + tabs(Am) * dtau);
      uk = un;
      if (done) break;
      if (it >= a.picard_max) { if (DIAG) diag[ST_PICARD_CAP]++; break; }
    }
    picard_its += it;
    u1 = uk;
  }
  const T xi1 = fma(T(0.5) * dtau, p.u + u1, p.xi);   // Eq. 9

  if (xi1 >= T(0) && xi1 <= T(1)) {
    // ---- O6: accept (inclusive, A-5).  The deposit of this sub-step is carried by xin.
    p.xi = xi1;
    p.u = u1;
    p.r -= dtau;
  } else {
    // ---- a4 / O7: crossing.  Land on the face the tentative step left through.
    const bool right = xi1 > T(1);
    const T dxi = right ? T(1) - p.xi : -p.xi;        // signed distance to that face
    const T Am = fma(T(0.5) * p.dA, dxi, A);          // A at the midpoint of the truncated step
    T D = fma(T(2) * Am, dxi, p.u * p.u);             // Eq. 12 (energy principle)
    if (DIAG && D < T(0)) diag[ST_NEG_DISC]++;
    D = tmax(D, T(0));
    const T sq = Prim<T>::sqrt(D);
    const T uc = right ? sq : -sq;
    // Root of F(dtau) = (A_m/2) dtau^2 + u dtau - dxi.  A-6: 2 dxi/(u+uc) when moving
    // towards the face, Eq. 13 (uc-u)/A_m otherwise; one reciprocal for both.
    const bool toward = right ? (p.u > T(0)) : (p.u < T(0));
    const T num = toward ? T(2) * dxi : uc - p.u;
    const T den = toward ? p.u + uc : Am;
    T dtc = Prim<T>::div(num, den);
    if (!toward && Am == T(0)) dtc = dtau;
    if (DIAG && !(dtc >= T(0) && dtc <= dtau)) diag[ST_CLAMPED]++;
    dtc = tmin(tmax(dtc, T(0)), dtau);                // NaN -> 0 (fmax/fmin drop the NaN)
    // a5 / O8: flush this cell visit, then enter the neighbour on its near face.
    deposit<T>(sJ, a.n_cells, p.c, p.xin, right ? T(1) : T(0));
    p.c = right ? ((p.c + 1 == a.n_cells) ? 0 : p.c + 1) : ((p.c == 0) ? a.n_cells - 1 : p.c - 1);
    p.xi = right ? T(0) : T(1);
    p.xin = p.xi;
    p.u = uc;
    p.r -= dtc;
    p.nc++;
    load_cell<T>(sA, a.n_cells, a.c_cap, p);
  }
  p.ns++;
}

template <typename T, bool CN_DIRECT, bool DIAG>
__global__ void __launch_bounds__(kBlock, 2) mover_kernel(const MoverArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* sJ = reinterpret_cast<double*>(smem_raw);                 // [n_cells] accumulators
  T* sA = reinterpret_cast<T*>(sJ + a.n_cells);                     // [n_cells] A on faces

  // ---- a0: field prologue.  E^{n+1/2} = (E^n + E^{n+1})/2 (north_star; A-11), A = (q/m)E/dx.
  for (int f = threadIdx.x; f < a.n_cells; f += blockDim.x) {
    sA[f] = (T)(a.qm_over_dx * (0.5 * (a.E_n[f] + a.E_np1[f])));
    sJ[f] = 0.0;
  }
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1u;
  long long next = 0, end = 0;       // warp-uniform: the warp's current index range
  bool exhausted = false;            // the global queue has run dry
  bool active = false;
  Lane<T> p;
  p.idx = -1;
  p.xi = p.u = p.r = p.AL = p.dA = p.cap = p.xin = T(0);
  p.c = 0; p.ns = p.nc = 0;
  unsigned long long tot_sub = 0, tot_cross = 0, tot_pic = 0;
  unsigned picard_its = 0;
  unsigned diag[ST_COUNT];
#pragma unroll
  for (int i = 0; i < ST_COUNT; ++i) diag[i] = 0;

  for (;;) {
    const unsigned parked = __ballot_sync(kFull, !active);
    if (parked) {
      const int n_parked = __popc(parked);
      // steady state: refill once enough lanes are parked; tail (queue dry): wait for all 32.
      const bool go = exhausted ? (n_parked == 32) : (n_parked >= a.refill_threshold);
      if (go) {
        if (next >= end && !exhausted) {
          // claim the next index range (a6: persistent-thread re-queue)
          unsigned long long t = 0;
          if (lane == 0) t = atomicAdd(a.queue, (unsigned long long)a.tile);
          t = __shfl_sync(kFull, t, 0);
          if ((long long)t >= a.n) { exhausted = true; }
          else { next = (long long)t; end = next + a.tile < a.n ? next + a.tile : a.n; }
        }
        if (!active) {
          // ---- a7: store the parked result (state n+1) ...
          if (p.idx >= 0) {
            deposit<T>(sJ, a.n_cells, p.c, p.xin, p.xi);   // last, partial cell visit
            if (a.xi1) {
              a.xi1[p.idx] = p.xi;
              a.v1[p.idx] = p.u * a.dx;
              a.cell1[p.idx] = p.c;
            }
            if (a.nsub_out) { a.nsub_out[p.idx] = p.ns; a.ncross_out[p.idx] = p.nc; }
            if (p.r > T(0)) diag[ST_SUBSTEP_CAP]++;        // cut off at max_substeps (A-9)
            tot_sub += p.ns; tot_cross += p.nc; tot_pic += picard_its;
            picard_its = 0;
            p.idx = -1;
          }
          // ---- a1: ... and load the next particle of the range, if any.
          const long long cand = next + __popc(parked & lt_mask);
          if (cand < end) {
            p.idx = cand;
            p.xi = a.xi0[cand];
            p.u = a.v0[cand] * a.inv_dx;
            p.c = a.cell0[cand];
            p.r = a.dt;
            p.xin = p.xi;
            p.ns = 0; p.nc = 0;
            load_cell<T>(sA, a.n_cells, a.c_cap, p);
            active = p.r > T(0);
          }
        }
        next = (next + n_parked < end) ? next + n_parked : end;
        if (exhausted && n_parked == 32) break;
      }
    }
    if (active) {
      substep<T, CN_DIRECT, DIAG>(a, sA, sJ, p, picard_its, diag);
      active = (p.r > T(0)) && (p.ns < (uint32_t)a.max_substeps);
    }
  }

  // ---- totals: warp reduce, one atomic per warp and slot.
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    tot_sub += __shfl_xor_sync(kFull, tot_sub, o);
    tot_cross += __shfl_xor_sync(kFull, tot_cross, o);
    tot_pic += __shfl_xor_sync(kFull, tot_pic, o);
  }
  if (lane == 0) {
    atomicAdd(&a.stats[ST_SUB], tot_sub);
    atomicAdd(&a.stats[ST_CROSS], tot_cross);
    if (tot_pic) atomicAdd(&a.stats[ST_PICARD_IT], tot_pic);
  }
#pragma unroll
  for (int i = ST_PICARD_CAP; i < ST_COUNT; ++i) {
    unsigned v = diag[i];
    v = __reduce_add_sync(kFull, v);
    if (lane == 0 && v) atomicAdd(&a.stats[i], (unsigned long long)v);
  }

  // ---- a8: one flush per block: scaled block sums -> this block's row of `partial`.
  __syncthreads();
  double* row = a.partial + (size_t)blockIdx.x * a.n_cells;
  for (int f = threadIdx.x; f < a.n_cells; f += blockDim.x) row[f] = a.scale * sJ[f];
}

}  // namespace picb200
