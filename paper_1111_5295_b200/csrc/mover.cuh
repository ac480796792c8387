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
//  * deposit, two modes (template PER_VISIT):
//      ENDPOINT (default): the per-sub-step linear-spline deposits of P:212 telescope exactly
//      (SURVEY P-7): J_f = G(X1 - f) - G(X0 - f), G = running integral of the hat function, X
//      unwrapped in cell units.  The sub-step loop only tracks k, the signed number of faces
//      crossed; at orbit end the particle adds +-1 to every face it passed completely (an int32
//      difference array in shared memory, native ATOMS.ADD, exact) and four fractional terms in
//      fp64.  The block prefix-sums the difference array once at its flush.
//      PER_VISIT: the paper's register accumulation: the stay in a cell from xi_in to
//      xi_out is flushed to the two faces on crossing / at orbit end with shared-memory fp64
//      atomics (a CAS loop on sm_100a: only 32-bit integer shared atomics are native).
//  * divergence (variable sub-step counts): persistent warps; a lane whose
//    orbit is finished parks its result and, once enough lanes of the warp are parked, the
//    parked lanes store and pull the next particles of the warp's current index range
//    (lane-level re-queue); ranges are claimed from a global counter.  With the state binned by
//    (cell, velocity class) the lanes of a warp run nearly the same sub-step and
//    crossing sequence, so both the crossing branch and the refill run with many lanes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pic_check.cuh"

namespace picb200 {

#ifndef PIC_BLOCK
#define PIC_BLOCK 384
#endif
constexpr int kBlock = PIC_BLOCK;  // threads per block
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
  int32_t tile;                // particles per claimed index range (multiple of 32), at most
  int32_t tile_min;            // ... and at least; in between: what is left / guide_div
  uint32_t guide_div;          // guided self-scheduling: 0 = always `tile`
  int32_t refill_threshold;    // parked lanes needed before a refill
  int32_t wrap_mask;           // n_cells - 1 if n_cells is a power of two, else 0
  int32_t deposit;             // 0 = VP variant: orbits only, no current deposit
  double qm_over_dx;           // (q/m)/dx
  T dx, inv_dx;
  T c_abs;                     // sqrt(2 eps_a / dx):   dtau_abs = c_abs / sqrt(|A| + |dA u|)
  T c_rel;                     // 2 eps_r:              dtau_rel = c_rel (|A|+|u|) / (|A|+|dA u|)
  T c_cap;                     // sqrt(4 kappa_max):    dtau_cap = c_cap / sqrt(|dA|)
  T dt, tol;
  double dt_exact;             // dt in fp64 (EXACT_T: the checkpointed remaining time starts here)
  double scale;                // w_q / dt : cell-unit deposit -> jbar contribution
  unsigned char* grid_scratch; // GGRID: [gridDim.x][grid_stride] bytes of global memory that stand in
  size_t grid_stride;          //        for the block's shared-memory grid (large n_cells)
  double* partial;             // [gridDim.x][n_cells] per-block sums (scaled)
  unsigned long long* queue;   // global index-range counter (zeroed before launch)
  unsigned long long* stats;   // [ST_COUNT] totals (accumulated)
};

// Dynamic shared memory of one block (bytes): F fp64 [n], A T [n+2] (halo), D int32 [n].
template <typename T>
__host__ __device__ inline size_t mover_smem_bytes(int n_cells) {
  size_t b = (size_t)n_cells * (sizeof(double) + sizeof(int32_t)) + (size_t)(n_cells + 2) * sizeof(T);
  return (b + 15) & ~(size_t)15;
}

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
  static __device__ __forceinline__ float rsqrt_est(float x) { return rsqrt(x); }
  static __device__ __forceinline__ float cap(float c, float absdA) { return c * rsqrt(absdA); }
  static __device__ __forceinline__ float div_unit(float a, float b) { return a * rcp(b); }
};

template <> struct Prim<double> {
  static __device__ __forceinline__ double rsqrt(double x) { return ::rsqrt(x); }  // 1 ulp
  static __device__ __forceinline__ double rcp(double x) { return 1.0 / x; }
  static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
  static __device__ __forceinline__ double div(double a, double b) { return a / b; }
  // Estimator only (Eq. 6-8 fix a step SIZE, not a state): MUFU.RSQ64H seed (2^-23) + one
  // Newton step -> relative error ~3e-14, 4 FP64 instructions instead of 5 + a slow-path test.
  // x = 0 or denormal gives NaN here (0 * inf); the caller's min/max then yield min(cap, r),
  // the same limit as A-1's floor on alpha.
  static __device__ __forceinline__ double rsqrt_est(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(0.5 * y, e, y);
  }
  // kappa cap c / sqrt(|dA|) (a step-size bound, like the estimator); |dA| = 0 -> +inf
  static __device__ __forceinline__ double cap(double c, double absdA) {
    return absdA > 0.0 ? c * rsqrt_est(absdA) : __longlong_as_double(0x7ff0000000000000LL);
  }
  // a / b for a normal, non-zero b (Eq. 11's denominator 1 - kappa in (0, 2) by A-2; the
  // crossing's u + u_c when moving towards the face): MUFU.RCP64H seed + two Newton steps, no
  // special-case path; <= 1.5 ulp.  A denormal b gives NaN, which the crossing clamp maps to 0.
  static __device__ __forceinline__ double div_unit(double a, double b) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(b));
    double e = fma(-b, y, 1.0);
    y = fma(y, e, y);
    e = fma(-b, y, 1.0);
    y = fma(y, e, y);
    return a * y;
  }
};

// xi in [0,1] (inclusive, A-5).  fp32: one unsigned compare of the bit pattern (non-negative
// floats order like their bits; a set sign bit or a NaN compares above 1.0f's pattern; -0.0 is
// rejected and then takes a zero-length crossing, A-5).
template <typename T> __device__ __forceinline__ bool in_unit(T x);
template <> __device__ __forceinline__ bool in_unit<float>(float x) {
  return __float_as_uint(x) <= 0x3f800000u; }
// fp64: the same test on the 64-bit pattern (two integer compares on the ALU pipe instead of two
// DSETP on the FP64 pipe, which bounds the fp64 kernel)
template <> __device__ __forceinline__ bool in_unit<double>(double x) {
  return (unsigned long long)__double_as_longlong(x) <= 0x3ff0000000000000ull; }

template <typename T> __device__ __forceinline__ T tabs(T x);
template <> __device__ __forceinline__ float tabs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double tabs<double>(double x) { return fabs(x); }
// min/max that drop a NaN in the FIRST operand (tmax(NaN, x) = x), which the estimator (A-1) and
// the crossing clamp rely on: fp32 uses the IEEE instructions (FMNMX, symmetric); fp64 a compare
// and select (DSETP + 2 SEL instead of the six-instruction IEEE fmin/fmax sequence).
template <typename T> __device__ __forceinline__ T tmin(T a, T b);
template <typename T> __device__ __forceinline__ T tmax(T a, T b);
template <> __device__ __forceinline__ float tmin<float>(float a, float b) { return fminf(a, b); }
template <> __device__ __forceinline__ float tmax<float>(float a, float b) { return fmaxf(a, b); }
template <> __device__ __forceinline__ double tmin<double>(double a, double b) { return a < b ? a : b; }
template <> __device__ __forceinline__ double tmax<double>(double a, double b) { return a > b ? a : b; }


// Tuning constants of the warp scheduler inside the kernel.
#ifndef PIC_KINNER
#define PIC_KINNER 64
#endif
#ifndef PIC_UNROLL
#define PIC_UNROLL 4
#endif
#ifndef PIC_REFILL
#define PIC_REFILL 4
#endif
#ifndef PIC_REFILL_VSORT
#define PIC_REFILL_VSORT 28
#endif
#ifndef PIC_MINBLOCKS_F32
#define PIC_MINBLOCKS_F32 3
#endif
constexpr int kGroup = PIC_UNROLL;        // sub-steps between two "any lane still in flight" votes
constexpr int kInner = PIC_KINNER;        // sub-step rounds between two refill votes
constexpr int kRefill = PIC_REFILL;       // parked lanes needed before a refill (cell binning)
constexpr int kRefillVsort = PIC_REFILL_VSORT;  // same with (cell, velocity class) binning

// Guided self-scheduling of the work queue: a warp claims `tile` particles while plenty are left
// and shrinking ranges (what is left / guide_div, never below tile_min) towards the end, so that
// the last ranges are short and the warps of the grid finish together.  `left` is the warp's own
// view (from the end of its last range), an over-estimate.
__device__ __forceinline__ uint32_t claim_size(int32_t tile, int32_t tile_min, uint32_t guide_div,
                                               uint32_t left) {
  if (guide_div == 0) return (uint32_t)tile;
  uint32_t w = (left / guide_div) & ~63u;
  w = w < (uint32_t)tile_min ? (uint32_t)tile_min : w;
  return w > (uint32_t)tile ? (uint32_t)tile : w;
}

// Per-lane particle registers.  r > 0 <=> an orbit is in flight.
template <typename T>
struct Lane {
  T xi, u, r;          // in-cell offset, velocity in cells/time, remaining time (O2)
  T AL, dA, cap;       // constants of the current cell (O3) and its kappa cap (A-2)
  T xa;                // ENDPOINT: xi at the orbit start;  PER_VISIT: xi at entry into the cell
  int32_t c;           // cell; with POW2 the UNWRAPPED cell c0 + k (wrapped by a mask on use)
  int32_t c0;          // ENDPOINT: start cell
  uint32_t ns, nc, nr; // sub-steps, crossings, crossings through a right face (k = 2 nr - nc;
                       // nr is not kept with POW2, where k = c - c0)
  uint32_t idx;        // particle index
  int32_t have;        // 0 = lane empty, 1 = a particle (in flight or parked), 2 = parked
                       // because it was cut off at max_substeps (A-9)
  T el;                // EXACT_T: time used since the last checkpoint (small, so its sums are
  double rem;          //          accurate); remaining time at the last checkpoint, exact
};

// EXACT_T (fp32 only): `r -= dtau` rounds to ulp(r)/2 at every sub-step, a random
// walk of ulp(dt) sqrt(n_sub)/2 in the integrated time (5e-5 at dt = 50 and 590 sub-steps: the
// particle is then moved for dt - 5e-5 and v is off by a * 5e-5).  With EXACT_T the time used is
// also summed in `el`, which stays below kGroup sub-steps and is therefore accurate to a few
// 1e-8, and every kGroup rounds the checkpoint `rem` (fp64) takes it over exactly and r is set
// to the correctly rounded remaining time again: r drifts for at most kGroup sub-steps and never
// accumulates.  r keeps its role (step limit, exact 0 at the orbit end).
template <typename T>
__device__ __forceinline__ void time_checkpoint(T& r, T& el, double& rem) {
  rem -= (double)el;
  el = T(0);
  // a parked lane (r = 0) stays parked whatever rounding left in rem; a negative remainder
  // (the orbit ran a few 1e-9 long) parks it
  r = (r > T(0)) ? tmax((T)rem, T(0)) : T(0);
}

// ENDPOINT: start-cell terms are collected in registers while consecutive particles of the lane
// start in the same cell (they do: the state is binned by cell) and flushed when it changes.
struct StartAcc {
  double f0, f1;       // pending contributions to faces cell, cell+1
  int32_t cell;        // -1 = empty
};

// O3: constants of cell c.  sA carries a one-face halo on both sides: sA[f+1] = A_f,
// sA[0] = A_{n-1}, sA[n+1] = A_0, so the two faces of cell c are sA[c+1], sA[c+2].
template <typename T>
__device__ __forceinline__ void load_cell(const T* __restrict__ sA, T c_cap, Lane<T>& p, int32_t c,
                                          int32_t n_cells) {
  c = chk(c, n_cells);
  const T AL = sA[c + 1], AR = sA[c + 2];
  p.AL = AL;
  p.dA = AR - AL;
  // A-2: dtau <= sqrt(4 kappa_max / |a'|); |dA| = 0 gives +inf (no cap).
  p.cap = Prim<T>::cap(c_cap, tabs(p.dA));
}

// PER_VISIT a5/O8: flush the stay [xin, xout] in cell c to the block accumulators.
template <typename T>
__device__ __forceinline__ void deposit_visit(double* __restrict__ sF, int32_t n_cells,
                                              int32_t c, T xin, T xout) {
  const T delta = xout - xin;
  const T right = delta * (T(0.5) * (xin + xout));
  const T left = delta - right;
  c = chk(c, n_cells);
  const int32_t cr = (c + 1 == n_cells) ? 0 : c + 1;
  atomicAdd(&sF[c], (double)left);
  atomicAdd(&sF[cr], (double)right);
}

__device__ __forceinline__ void flush_start(double* __restrict__ sF, int32_t n, StartAcc& s) {
  if (s.cell >= 0) {
    s.cell = chk(s.cell, n);
    atomicAdd(&sF[s.cell], s.f0);
    atomicAdd(&sF[(s.cell + 1 == n) ? 0 : s.cell + 1], s.f1);
  }
  s.cell = -1;
  s.f0 = s.f1 = 0.0;
}

// ENDPOINT a5/O8 (SURVEY P-7): J_f = G(X1 - f) - G(X0 - f) for a particle that went from
// (c0, x0) to (c1, x1) crossing k faces (signed).  With g0(x) = 1 - (1-x)^2/2 (own left face)
// and g1(x) = x^2/2 (own right face):
//   J_f = [faces passed completely: +-1] + g0(x1)[f=c1] + g1(x1)[f=c1+1]
//                                       - g0(x0)[f=c0] - g1(x0)[f=c0+1].
// The +-1 run covers faces [c0, c0+k) for k > 0 and [c1, c1+|k|) for k < 0 (periodic); it goes
// into the difference array sD (prefix-summed at the block flush), whole turns of the ring into
// sD[0].  Start-cell terms go through the lane's register accumulator.
// End-cell terms are handed back (e0 on face c1, e1 on face c1+1; `pending` set) so that the warp
// can add up the lanes that end in the same cell before touching shared memory.
struct EndTerms {
  double e0, e1;
  int32_t cell;
  bool pending;
};

__device__ __forceinline__ void deposit_endpoint(double* __restrict__ sF, int32_t* __restrict__ sD,
                                                 int32_t n, StartAcc& acc, EndTerms& et, int32_t c0,
                                                 double x0, int32_t c1, double x1, int32_t k) {
  if (c0 != acc.cell) {
    flush_start(sF, n, acc);
    acc.cell = c0;
  }
  if (k == 0) {
    // same cell: one term per face, no cancellation between large numbers
    const double d = x1 - x0, m = 0.5 * (x0 + x1);
    acc.f0 += d * (1.0 - m);
    acc.f1 += d * m;
    return;
  }
  acc.f0 += 0.5 * (1.0 - x0) * (1.0 - x0) - 1.0;
  acc.f1 -= 0.5 * x0 * x0;
  et.e0 = 1.0 - 0.5 * (1.0 - x1) * (1.0 - x1);
  et.e1 = 0.5 * x1 * x1;
  et.cell = c1;
  et.pending = true;
  const int32_t sgn = k > 0 ? 1 : -1;
  int32_t len = k > 0 ? k : -k;
  const int32_t a = k > 0 ? c0 : c1;
  if (len >= n) {
    const int32_t w = len / n;
    len -= w * n;
    atomicAdd(&sD[0], sgn * w);
  }
  if (len > 0) {
    const int32_t e = a + len;
    atomicAdd(&sD[chk(a, n)], sgn);
    if (e < n) atomicAdd(&sD[chk(e, n)], -sgn);
    else if (e > n) { atomicAdd(&sD[0], sgn); atomicAdd(&sD[chk(e - n, n)], -sgn); }
  }
}

// Warp-uniform: add the pending end-cell terms of all lanes to the block accumulators, one pair
// of shared-memory atomics per DISTINCT end cell (lanes of a warp mostly end in the same one or
// two cells, and the fp64 shared atomic is a CAS loop that would serialise them).
__device__ __forceinline__ void warp_deposit_end(double* __restrict__ sF, int32_t n, int lane,
                                                 const EndTerms& et) {
  unsigned todo = __ballot_sync(kFull, et.pending);
  bool mine_left = et.pending;
  // up to two shared end cells are summed across the warp ...
#pragma unroll 1
  for (int it = 0; it < 2 && todo; ++it) {
    const int leader = __ffs(todo) - 1;
    const int32_t key = __shfl_sync(kFull, et.cell, leader);
    const bool mine = mine_left && et.cell == key;
    const unsigned grp = __ballot_sync(kFull, mine);
    todo &= ~grp;
    if (__popc(grp) == 1) continue;              // a singleton goes the direct way below
    double a = mine ? et.e0 : 0.0, b = mine ? et.e1 : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_xor_sync(kFull, a, o);
      b += __shfl_xor_sync(kFull, b, o);
    }
    if (lane == leader) {
      (void)chk(key, n);
      atomicAdd(&sF[key], a);
      atomicAdd(&sF[(key + 1 == n) ? 0 : key + 1], b);
    }
    if (mine) mine_left = false;
  }
  // ... lanes that end anywhere else (long, scattered orbits) add their own terms
  if (mine_left) {
    (void)chk(et.cell, n);
    atomicAdd(&sF[et.cell], et.e0);
    atomicAdd(&sF[(et.cell + 1 == n) ? 0 : et.cell + 1], et.e1);
  }
}

// Warp-uniform: the lanes flagged in `flush` hand their start-cell accumulators to the block
// sums.  Lanes of a warp walk through the binned particle list together, so they leave a start
// cell in the same refill: flushed one by one inside deposit_endpoint, 32 lanes hit the same two
// addresses with the CAS loop of the shared fp64 add and spin ~30 rounds each (42 % of the
// instructions of a 2 M ion pass, profiles/r2_bench.md); summed over the warp first it is one add
// per face.
__device__ __forceinline__ void warp_flush_start(double* __restrict__ sF, int32_t n, int lane,
                                                 StartAcc& acc, bool flush) {
  if (!__any_sync(kFull, flush)) return;
  EndTerms t;
  t.e0 = acc.f0; t.e1 = acc.f1; t.cell = flush ? acc.cell : 0; t.pending = flush;
  warp_deposit_end(sF, n, lane, t);
  if (flush) { acc.cell = -1; acc.f0 = acc.f1 = 0.0; }
}

// ---- a8: one flush per block.  Inclusive prefix sum of the difference array over the
// faces (each thread owns a contiguous chunk), then scaled block sums -> this block's row of
// `partial`.  Called by every thread of the block after its warps have left the particle loop.
template <typename T>
__device__ __forceinline__ void block_flush(const MoverArgs<T>& a, const double* __restrict__ sF,
                                            const int32_t* __restrict__ sD, int32_t* s_wtot) {
  const int lane = threadIdx.x & 31;
  __syncthreads();
  const int per = (a.n_cells + (int)blockDim.x - 1) / (int)blockDim.x;
  const int fb = min((int)threadIdx.x * per, a.n_cells), fe = min(fb + per, a.n_cells);
  int32_t s = 0;
  for (int f = fb; f < fe; ++f) s += sD[f];
  int32_t inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int32_t t = __shfl_up_sync(kFull, inc, o);
    if (lane >= o) inc += t;
  }
  const int wid = threadIdx.x >> 5;
  if (lane == 31) s_wtot[wid] = inc;
  __syncthreads();
  int32_t run = inc - s;                       // exclusive within the warp
  for (int w = 0; w < wid; ++w) run += s_wtot[w];
  double* row = a.partial + (size_t)blockIdx.x * a.n_cells;
  for (int f = fb; f < fe; ++f) {
    run += sD[f];
    row[f] = a.scale * (sF[f] + (double)run);
  }
}

// The same flush for the GGRID instantiation, whose "shared" grid copy is a row of GLOBAL memory
// that the block's warps have been updating with atomics (performed in L2).  Two differences:
// the faces are taken in tiles of blockDim.x with thread t on face base + t, so that a warp reads
// and writes 32 consecutive elements (contiguous per-thread chunks cost one memory transaction
// per lane), with a running carry from tile to tile; and sF / sD are read with ld.global.cg
// (__ldcg, L2), never through a possibly stale L1 line or a read-only path.  (The __restrict__
// qualifiers of the helpers above only promise that nothing else writes the arrays while that
// helper runs, which holds; the compiler does not turn them into non-coherent loads -- no
// LDG.CONSTANT in any mover_kernel instantiation -- but this path does not depend on it.)
template <typename T>
__device__ __forceinline__ void block_flush_global(const MoverArgs<T>& a, const double* sF,
                                                   const int32_t* sD, int32_t* s_wtot) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (int)blockDim.x >> 5;
  __syncthreads();
  double* row = a.partial + (size_t)blockIdx.x * a.n_cells;
  int32_t carry = 0;                             // sum of sD over the faces of earlier tiles
  for (int base = 0; base < a.n_cells; base += (int)blockDim.x) {
    const int f = base + (int)threadIdx.x;
    const int32_t d = f < a.n_cells ? __ldcg(sD + f) : 0;
    int32_t inc = d;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int32_t t = __shfl_up_sync(kFull, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_wtot[wid] = inc;
    __syncthreads();
    int32_t run = carry + inc, tot = 0;          // inclusive prefix sum up to face f
    for (int w = 0; w < nw; ++w) {
      const int32_t t = s_wtot[w];
      if (w < wid) run += t;
      tot += t;
    }
    if (f < a.n_cells) row[f] = a.scale * (__ldcg(sF + f) + (double)run);
    carry += tot;
    __syncthreads();                             // s_wtot is rewritten by the next tile
  }
}

// One sub-step (O3-O8) of the lane's particle: estimate dtau, tentative Crank-Nicolson step in
// the current cell, accept it if it stays in the cell, otherwise truncate it at the face.
// CN_DIRECT: Eq. 11, else Picard on Eq. 9-10.  The max_substeps cap (A-9) is checked by the
// caller once every kInner sub-steps.
template <typename T, bool CN_DIRECT, bool DIAG, bool PER_VISIT, bool POW2, bool EXACT_T>
__device__ __forceinline__ void substep(const MoverArgs<T>& a, const T* __restrict__ sA,
                                        double* __restrict__ sF, Lane<T>& p,
                                        unsigned& picard_its, unsigned* diag) {
  // ---- a2 / O4: estimator (Eq. 6-8), L1 form, in cell units:
  //   alpha = dx (|A| + |dA u|)/2, beta = eps_r dx (|A| + |u|)
  //   dtau = max( sqrt(eps_a/alpha), beta/alpha ) = max( c_abs d, c_rel (|A|+|u|) d^2 ),
  //   d = (|A| + |dA u|)^(-1/2)  (one rsqrt).
  // A-1 (alpha = 0): d = +inf, the first term is +inf and the second +inf or NaN; the IEEE
  // max/min drop the NaN, so dtau = min(cap, r) -- the same limit as flooring alpha.
  const bool live = p.r > T(0);   // counters below count orbits in flight, not parked lanes
  const T A = fma(p.dA, p.xi, p.AL);
  const T absA = tabs(A);
  const T d = Prim<T>::rsqrt_est(absA + tabs(p.dA * p.u));
  T dtau = tmax((a.c_rel * (absA + tabs(p.u))) * d, a.c_abs) * d;
  if (DIAG && live && dtau > p.cap) diag[ST_KAPPA_CAP]++;
  dtau = tmin(tmin(dtau, p.cap), p.r);

  // ---- a3 / O5: Crank-Nicolson step over dtau with the linear field of the current cell (A-4).
  const T h = T(0.5) * dtau;
  T u1;
  if (CN_DIRECT) {
    // Eq. 11: kappa = a' dtau^2/4;  u' = [A dtau + (1+kappa) u] / (1-kappa).
    const T kappa = p.dA * (h * h);
    const T num = fma(A, dtau, fma(kappa, p.u, p.u));
    u1 = Prim<T>::div_unit(num, T(1) - kappa);
  } else {
    // Picard (A-3): u' <- u; u'' = u + dtau A(xi + dtau (u+u')/4) until
    // |u''-u'| <= tol (|u''| + |A_m| dtau).
    T uk = p.u;
    int it = 0;
    for (;;) {
      const T xim = fma(T(0.5) * h, p.u + uk, p.xi);
      const T Am = fma(p.dA, xim, p.AL);
      const T un = fma(dtau, Am, p.u);
      ++it;
      const bool done = tabs(un - uk) <= a.tol * (tabs(un) + tabs(Am) * dtau);
      uk = un;
      if (done) break;
      if (it >= a.picard_max) { if (DIAG && live) diag[ST_PICARD_CAP]++; break; }
    }
    if (live) picard_its += it;
    u1 = uk;
  }
  const T xi1 = fma(h, p.u + u1, p.xi);               // Eq. 9
  // exact per-particle sub-step count only in the counting build (DIAG); a parked lane (r = 0)
  // takes a zero-length step that changes nothing and is not counted
  if (DIAG) { if (live) p.ns++; }

  if (in_unit<T>(xi1)) {
    // ---- O6: accept (inclusive, A-5).
    p.xi = xi1;
    p.u = u1;
    p.r -= dtau;
    if (EXACT_T) p.el += dtau;
  } else {
    // ---- a4 / O7: crossing.  Land on the face the tentative step left through.
    const bool right = xi1 > T(1);
    const T face = right ? T(1) : T(0);
    const T dxi = face - p.xi;                        // signed distance to that face
    const T Am = fma(T(0.5) * p.dA, dxi, A);          // A at the midpoint of the truncated step
    T D = fma(Am + Am, dxi, p.u * p.u);               // Eq. 12 (energy principle)
    if (DIAG && D < T(0)) diag[ST_NEG_DISC]++;
    D = tmax(D, T(0));
    const T sq = Prim<T>::sqrt(D);
    const T uc = right ? sq : -sq;
    // Root of F(dtau) = (A_m/2) dtau^2 + u dtau - dxi.  A-6: 2 dxi/(u+uc) when moving
    // towards the face (the common case), Eq. 13 (uc-u)/A_m otherwise.
    const bool toward = (right ? p.u : -p.u) > T(0);
    T dtc;
    if (toward) {
      dtc = Prim<T>::div_unit(dxi + dxi, p.u + uc);   // |u + uc| >= |u| > 0
    } else {
      dtc = (Am == T(0)) ? dtau : Prim<T>::div(uc - p.u, Am);
    }
    if (DIAG && !(dtc >= T(0) && dtc <= dtau)) diag[ST_CLAMPED]++;
    dtc = tmin(tmax(dtc, T(0)), dtau);                // NaN -> 0 (IEEE max/min drop the NaN)
    // a5: PER_VISIT flushes this cell visit now; ENDPOINT only counts the face.
    // enter the neighbour on its near face
    int32_t cw;                                       // wrapped index of the new cell
    if (POW2) {
      if (PER_VISIT) deposit_visit<T>(sF, a.n_cells, p.c & a.wrap_mask, p.xa, face);
      p.c += right ? 1 : -1;                          // unwrapped: k = c - c0
      cw = p.c & a.wrap_mask;
    } else {
      if (PER_VISIT) deposit_visit<T>(sF, a.n_cells, p.c, p.xa, face);
      int32_t cn = p.c + (right ? 1 : -1);
      cn = (cn == a.n_cells) ? 0 : cn;
      cn = (cn < 0) ? a.n_cells - 1 : cn;
      p.c = cn;
      cw = cn;
      if (right) p.nr++;
    }
    // crossings are counted per particle where something needs them: the counting build, and
    // k = 2 nr - nc of a non-power-of-two grid
    if (DIAG || !POW2) p.nc++;
    p.xi = T(1) - face;
    if (PER_VISIT) p.xa = p.xi;
    p.u = uc;
    p.r -= dtc;
    if (EXACT_T) p.el += dtc;
    load_cell<T>(sA, a.c_cap, p, cw, a.n_cells);
  }
}

// Launch shape per precision: fp32 384 threads x 3 blocks/SM (56 registers); fp64 512 threads x
// 2 blocks/SM (64 registers -> 32 warps/SM instead of 24 with 384-thread blocks).
#ifndef PIC_BLOCK_F64
#define PIC_BLOCK_F64 512
#endif
template <typename T> struct LaunchCfg {
  static constexpr int min_blocks = 2;
  static constexpr int block = PIC_BLOCK_F64;
};
template <> struct LaunchCfg<float> {
  static constexpr int min_blocks = PIC_MINBLOCKS_F32;
  static constexpr int block = kBlock;
};

// GGRID: the per-block copy of the grid (field faces, fp64 sums, difference array) lives in
// global memory instead of shared memory -- the fallback for grids whose n_cells (8 + 4 +
// sizeof(T)) bytes exceed the 227 KB a block can have (S7 hard part 6).  The field is read
// through L1/L2 and the deposits are global atomics on the block's own (L2-resident) row.
template <typename T, bool CN_DIRECT, bool DIAG, bool PER_VISIT, bool POW2, bool EXACT_T = false,
          bool GGRID = false>
__global__ void __launch_bounds__(LaunchCfg<T>::block, LaunchCfg<T>::min_blocks)
mover_kernel(const MoverArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  unsigned char* smem_raw = GGRID ? a.grid_scratch + (size_t)blockIdx.x * a.grid_stride : smem_dyn;
  double* sF = reinterpret_cast<double*>(smem_raw);                 // [n] fp64 accumulators
  T* sA = reinterpret_cast<T*>(sF + a.n_cells);                     // [n+2] A on faces + halo
  int32_t* sD = reinterpret_cast<int32_t*>(sA + a.n_cells + 2);     // [n] difference array
  __shared__ int32_t s_wtot[LaunchCfg<T>::block / 32];

  // ---- a0: field prologue.  E^{n+1/2} = (E^n + E^{n+1})/2 (north_star; A-11), A = (q/m)E/dx.
  for (int f = threadIdx.x; f < a.n_cells; f += blockDim.x) {
    const T Af = (T)(a.qm_over_dx * (0.5 * (a.E_n[f] + a.E_np1[f])));
    sA[f + 1] = Af;
    if (f == 0) sA[a.n_cells + 1] = Af;
    if (f == a.n_cells - 1) sA[0] = Af;
    sF[f] = 0.0;
    sD[f] = 0;
  }
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1u;
  const uint32_t n32 = (uint32_t)a.n;
  uint32_t next = 0, end = 0;        // warp-uniform: the warp's current index range
  bool exhausted = false;            // the global queue has run dry
  Lane<T> p;
  p.have = 0;
  p.idx = 0;
  p.xi = p.u = p.r = p.AL = p.dA = p.cap = p.xa = p.el = T(0);
  p.rem = 0.0;
  p.c = p.c0 = 0; p.ns = p.nc = p.nr = 0;
  StartAcc acc;
  acc.cell = -1; acc.f0 = acc.f1 = 0.0;
  unsigned long long tot_sub = 0, tot_cross = 0, tot_pic = 0;
  unsigned picard_its = 0;
  unsigned diag[ST_COUNT];
#pragma unroll
  for (int i = 0; i < ST_COUNT; ++i) diag[i] = 0;

  for (;;) {
    // A-9: an orbit that has used max_substeps with time left is parked with r < 0 (checked
    // once per kInner sub-steps, so it may overshoot the cap by fewer than kInner).
    if (p.ns >= (uint32_t)a.max_substeps && p.r > T(0)) { p.r = T(0); p.have = 2; }

    // ---- a6/a7/a1: lane-level re-queue.  Parked lanes (r <= 0) wait until enough of them have
    // gathered, then store their result and pull the next particles of the warp's range.
    const unsigned parked = __ballot_sync(kFull, !(p.r > T(0)));
    if (parked) {
      const int n_parked = __popc(parked);
      // steady state: refill once enough lanes are parked; tail (queue dry): wait for all 32.
      const bool go = exhausted ? (n_parked == 32) : (n_parked >= a.refill_threshold);
      if (go) {
        if (next >= end && !exhausted) {
          // claim the next index range (persistent-thread re-queue)
          const uint32_t want = claim_size(a.tile, a.tile_min, a.guide_div, n32 - end);
          unsigned long long t = 0;
          if (lane == 0) t = atomicAdd(a.queue, (unsigned long long)want);
          t = __shfl_sync(kFull, t, 0);
          if (t >= (unsigned long long)a.n) { exhausted = true; }
          else {
            next = (uint32_t)t;
            end = (n32 - next > want) ? next + want : n32;
          }
        }
        EndTerms et;
        et.pending = false; et.cell = 0; et.e0 = et.e1 = 0.0;
        if (!PER_VISIT)
          warp_flush_start(sF, a.n_cells, lane, acc,
                           !(p.r > T(0)) && p.have && a.deposit && acc.cell >= 0 && p.c0 != acc.cell);
        if (!(p.r > T(0))) {
          // ---- a7: store the parked result (state n+1) and deposit its current ...
          if (p.have) {
            // canonical end cell and signed face count
            const int32_t c1 = POW2 ? (p.c & a.wrap_mask) : p.c;
            const int32_t k = POW2 ? (p.c - p.c0) : (int32_t)(2u * p.nr - p.nc);
            if (PER_VISIT) deposit_visit<T>(sF, a.n_cells, c1, p.xa, p.xi);
            else if (a.deposit)
              deposit_endpoint(sF, sD, a.n_cells, acc, et, p.c0, (double)p.xa, c1, (double)p.xi, k);
            p.c = c1;
            p.idx = chk(p.idx, a.n);
            if (a.xi1) {
              a.xi1[p.idx] = p.xi;
              a.v1[p.idx] = p.u * a.dx;
              a.cell1[p.idx] = p.c;
            }
            if (a.nsub_out) { a.nsub_out[p.idx] = p.ns; a.ncross_out[p.idx] = p.nc; }
            if (p.have == 2) diag[ST_SUBSTEP_CAP]++;       // cut off at max_substeps (A-9)
            tot_sub += p.ns; tot_cross += p.nc; tot_pic += picard_its;
            picard_its = 0;
            p.have = 0;
            p.r = T(0);
            p.ns = 0;
          }
          // ---- a1: ... and load the next particle of the range, if any.
          const uint32_t rank = (uint32_t)__popc(parked & lt_mask);
          if (rank < end - next) {
            const uint32_t cand = chk(next + rank, a.n);
            p.idx = cand;
            p.have = 1;
            p.xi = a.xi0[cand];
            p.u = a.v0[cand] * a.inv_dx;
            p.c = a.cell0[cand];
            p.r = a.dt;
            if (EXACT_T) { p.rem = a.dt_exact; p.el = T(0); }
            p.xa = p.xi;
            p.c0 = p.c;
            p.ns = 0; p.nc = 0; p.nr = 0;
            load_cell<T>(sA, a.c_cap, p, p.c, a.n_cells);
          }
        }
        if (!PER_VISIT) warp_deposit_end(sF, a.n_cells, lane, et);
        next = ((uint32_t)n_parked < end - next) ? next + (uint32_t)n_parked : end;
        if (exhausted && n_parked == 32) break;
      }
    }

    // ---- kInner sub-steps of every lane that has an orbit in flight
    // Every lane steps: with r = 0 (parked or empty) dtau = 0, the tentative step reproduces
    // (xi, u) bit for bit and is accepted, so no per-lane guard branch is needed; the warp leaves
    // the rounds early once no lane has an orbit in flight (checked every kGroup sub-steps).
#pragma unroll 1
    for (int j = 0; j < kInner / kGroup; ++j) {
      // fast build: sub-steps are counted per group of kGroup rounds (an upper bound, less than
      // kGroup above the exact count per particle); it feeds the A-9 cap and pic_stats.n_sub
      if (!DIAG) { if (p.r > T(0)) p.ns += kGroup; }
#pragma unroll
      for (int g = 0; g < kGroup; ++g)
        substep<T, CN_DIRECT, DIAG, PER_VISIT, POW2, EXACT_T>(a, sA, sF, p, picard_its, diag);
      if (EXACT_T) time_checkpoint<T>(p.r, p.el, p.rem);
      if (!__any_sync(kFull, p.r > T(0))) break;
    }
  }
  if (!PER_VISIT) flush_start(sF, a.n_cells, acc);

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

  if constexpr (GGRID) block_flush_global<T>(a, sF, sD, s_wtot);
  else block_flush<T>(a, sF, sD, s_wtot);
}

}  // namespace picb200
