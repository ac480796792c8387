// mover2.cuh — the fp32 production instantiation of the mover (a0..a8) with TWO
// particles per lane and packed FP32 arithmetic (sm_100a FFMA2 / FMUL2 / FADD2).
//
// Why: mover_kernel<float> is bound by instruction issue (90 % of the issue slots busy, FMA pipe
// 47 %, profiles/r2_mover_ncu.md).  sm_100a executes fma/mul/add.f32x2 on a register pair as ONE
// issued instruction (measured with pic_microbench, profiles/r2_microbench.md: the same FMA-pipe
// time as two scalar FFMAs with half the instructions).  The estimator (Eq. 6-8) and the
// Crank-Nicolson update (Eq. 11) of two independent particles are the same straight-line
// arithmetic, so each lane carries two orbits ("slots" .x and .y of float2 registers) and runs
// them through packed instructions; abs/min/max/MUFU stay scalar.  The crossing (Eq. 12-13,
// P:184-206) is handled per slot, only by the lanes whose slot left its cell.
//
// Arithmetic, operation order and rounding are those of mover_kernel<float, direct, fast build,
// end-point deposit, power-of-two grid>: the two kernels produce bit-identical orbits (tested).
// Everything else (lane-level re-queue, end-point deposit, block flush) is shared with mover.cuh;
// the warp now re-queues 64 slots instead of 32 lanes.
//
// Per-cell constants {A_L, dA, kappa cap} are precomputed once per block into a float4 table
// (three loads on cell entry instead of two loads + FADD + MUFU.RSQ + FMUL): 28 B of shared memory
// per cell, two 512-thread blocks per SM (64 registers per thread, 32 warps = 2,048 orbits per SM).
#pragma once
#include "mover.cuh"

namespace picb200 {

#ifndef PIC_REFILL2
#define PIC_REFILL2 8
#endif
#ifndef PIC_REFILL2_VSORT
#define PIC_REFILL2_VSORT 56
#endif
#ifndef PIC_BLOCK2
#define PIC_BLOCK2 512
#endif
constexpr int kBlock2 = PIC_BLOCK2;               // threads per block of mover2_kernel
constexpr int kRefill2 = PIC_REFILL2;             // parked slots (of 64) needed before a refill
constexpr int kRefill2Vsort = PIC_REFILL2_VSORT;  // same with phase-space binning

// Dynamic shared memory of one block: F fp64 [n], C float4 [n] {A_L, dA, cap, -}, D int32 [n].
__host__ __device__ inline size_t mover2_smem_bytes(int n_cells) {
  return (size_t)n_cells * (sizeof(double) + sizeof(float4) + sizeof(int32_t));
}

// Three scalar shared-memory loads of one table entry (inline PTX so that they are not merged
// into one LDS.128: the values go straight into one slot's halves of the packed register pairs,
// a vector load would need moves on the common path).
__device__ __forceinline__ void load_cell3(const float4* cc, float& AL, float& dA, float& cap) {
  const unsigned addr = (unsigned)__cvta_generic_to_shared(cc);
  asm volatile("ld.volatile.shared.f32 %0, [%1];" : "=f"(AL) : "r"(addr) : "memory");
  asm volatile("ld.volatile.shared.f32 %0, [%1+4];" : "=f"(dA) : "r"(addr) : "memory");
  asm volatile("ld.volatile.shared.f32 %0, [%1+8];" : "=f"(cap) : "r"(addr) : "memory");
}

template <int S> __device__ __forceinline__ float get(const float2& v) { return S ? v.y : v.x; }
template <int S> __device__ __forceinline__ void put(float2& v, float x) { if (S) v.y = x; else v.x = x; }

// Per-lane registers: slot 0 in .x / [0], slot 1 in .y / [1].  r > 0 <=> an orbit is in flight.
struct Lane2 {
  float2 xi, u, r;       // in-cell offset, velocity in cells/time, remaining time (O2)
  float2 AL, dA, cap;    // constants of the slot's current cell (O3) and its kappa cap (A-2)
  float xa[2];           // xi at the orbit start
  int32_t c[2], c0[2];   // unwrapped cell c0 + k, start cell
  uint32_t ns[2], idx[2];
  int32_t have[2];       // 0 = empty, 1 = a particle, 2 = cut off at max_substeps (A-9)
};

// a4 / O7 for slot S: the tentative step left the cell; land on that face.
template <int S>
__device__ __forceinline__ void cross2(const MoverArgs<float>& a, const float4* __restrict__ sC,
                                       Lane2& p, const float2& A2, const float2& dtau2,
                                       float2& nxi, float2& nu, float2& used) {
  const float xi = get<S>(p.xi), u = get<S>(p.u), dA = get<S>(p.dA);
  const float A = get<S>(A2), dtau = get<S>(dtau2);
  const bool right = get<S>(nxi) > 1.0f;
  const float face = right ? 1.0f : 0.0f;
  const float dxi = face - xi;                          // signed distance to that face
  const float Am = fmaf(0.5f * dA, dxi, A);             // A at the midpoint of the truncated step
  float D = fmaf(Am + Am, dxi, u * u);                  // Eq. 12 (energy principle)
  D = fmaxf(D, 0.0f);
  const float sq = Prim<float>::sqrt(D);
  const float uc = right ? sq : -sq;
  // Root of (A_m/2) dtau^2 + u dtau - dxi; A-6: 2 dxi/(u+uc) when moving towards the
  // face, Eq. 13 (uc-u)/A_m otherwise.
  const bool toward = (right ? u : -u) > 0.0f;
  float dtc;
  if (toward) dtc = Prim<float>::div(dxi + dxi, u + uc);
  else dtc = (Am == 0.0f) ? dtau : Prim<float>::div(uc - u, Am);
  dtc = fminf(fmaxf(dtc, 0.0f), dtau);                  // NaN -> 0
  p.c[S] += right ? 1 : -1;                             // unwrapped: k = c - c0
  put<S>(nxi, 1.0f - face);
  put<S>(nu, uc);
  put<S>(used, dtc);
  float nAL, ndA, ncap;
  load_cell3(sC + chk(p.c[S] & a.wrap_mask, a.n_cells), nAL, ndA, ncap);
  put<S>(p.AL, nAL);
  put<S>(p.dA, ndA);
  put<S>(p.cap, ncap);
}

// One sub-step (O3-O8) of both slots.  A parked or empty slot has r = 0, so dtau = 0 and the
// tentative step reproduces (xi, u) bit for bit and is accepted (no per-slot guard).
__device__ __forceinline__ void substep2(const MoverArgs<float>& a, const float4* __restrict__ sC,
                                         Lane2& p) {
  const float2 half2 = make_float2(0.5f, 0.5f), one2 = make_float2(1.0f, 1.0f),
               mone2 = make_float2(-1.0f, -1.0f), crel2 = make_float2(a.c_rel, a.c_rel);
  // ---- a2 / O4: estimator (Eq. 6-8), cell units, one rsqrt per slot
  const float2 A = __ffma2_rn(p.dA, p.xi, p.AL);
  const float2 t = __fmul2_rn(p.dA, p.u);
  float2 s, w, d;
  s.x = fabsf(A.x) + fabsf(t.x);
  s.y = fabsf(A.y) + fabsf(t.y);
  w.x = fabsf(A.x) + fabsf(p.u.x);
  w.y = fabsf(A.y) + fabsf(p.u.y);
  d.x = Prim<float>::rsqrt(s.x);
  d.y = Prim<float>::rsqrt(s.y);
  w = __fmul2_rn(__fmul2_rn(w, crel2), d);
  w.x = fmaxf(a.c_abs, w.x);                            // A-1: a NaN (0 * inf) is dropped
  w.y = fmaxf(a.c_abs, w.y);
  float2 dtau = __fmul2_rn(w, d);
  dtau.x = fminf(fminf(dtau.x, p.cap.x), p.r.x);        // A-2 cap, remaining time
  dtau.y = fminf(fminf(dtau.y, p.cap.y), p.r.y);
  // ---- a3 / O5: Eq. 11 with h = dtau/2: kappa = a' h^2, u' = [A dtau + (1+kappa)u]/(1-kappa)
  const float2 h = __fmul2_rn(dtau, half2);
  const float2 kap = __fmul2_rn(p.dA, __fmul2_rn(h, h));
  const float2 num = __ffma2_rn(A, dtau, __ffma2_rn(kap, p.u, p.u));
  const float2 den = __ffma2_rn(kap, mone2, one2);
  float2 rd;
  rd.x = Prim<float>::rcp(den.x);
  rd.y = Prim<float>::rcp(den.y);
  float2 nu = __fmul2_rn(num, rd);
  float2 nxi = __ffma2_rn(h, __fadd2_rn(p.u, nu), p.xi);  // Eq. 9
  float2 used = dtau;
  // ---- O6 / O7: accept both (inclusive, A-5), or truncate the slots that left their cell
  const bool ok0 = in_unit<float>(nxi.x), ok1 = in_unit<float>(nxi.y);
  // (behind a warp-uniform vote: the divergent per-slot blocks then sit inside a uniform branch)
  if (__any_sync(kFull, !(ok0 && ok1))) {
    if (!ok0) cross2<0>(a, sC, p, A, dtau, nxi, nu, used);
    if (!ok1) cross2<1>(a, sC, p, A, dtau, nxi, nu, used);
  }
  p.xi = nxi;
  p.u = nu;
  p.r = __ffma2_rn(used, mone2, p.r);
}

// a7 + a1 for slot S of a parked lane: store the finished orbit (state n+1), deposit its current
// (end-point form), then load the next particle of the warp's range, if any.
template <int S>
__device__ __forceinline__ void refill_slot(const MoverArgs<float>& a, double* __restrict__ sF,
                                            int32_t* __restrict__ sD, const float4* __restrict__ sC,
                                            Lane2& p, StartAcc& acc, EndTerms& et, uint32_t rank,
                                            uint32_t next, uint32_t end,
                                            unsigned long long& tot_sub, unsigned& capped) {
  et.pending = false; et.cell = 0; et.e0 = et.e1 = 0.0;
  if (get<S>(p.r) > 0.0f) return;
  if (p.have[S]) {
    const int32_t c1 = p.c[S] & a.wrap_mask;
    const int32_t k = p.c[S] - p.c0[S];
    const float xi = get<S>(p.xi);
    if (a.deposit)
      deposit_endpoint(sF, sD, a.n_cells, acc, et, p.c0[S], (double)p.xa[S], c1, (double)xi, k);
    p.idx[S] = chk(p.idx[S], a.n);
    if (a.xi1) {
      a.xi1[p.idx[S]] = xi;
      a.v1[p.idx[S]] = get<S>(p.u) * a.dx;
      a.cell1[p.idx[S]] = c1;
    }
    if (p.have[S] == 2) capped++;
    tot_sub += p.ns[S];
    p.have[S] = 0;
    put<S>(p.r, 0.0f);
    p.ns[S] = 0;
  }
  if (rank < end - next) {
    const uint32_t cand = chk(next + rank, a.n);
    p.idx[S] = cand;
    p.have[S] = 1;
    const float xi = a.xi0[cand];
    const int32_t c = chk(a.cell0[cand], a.n_cells);
    put<S>(p.xi, xi);
    put<S>(p.u, a.v0[cand] * a.inv_dx);
    put<S>(p.r, a.dt);
    p.xa[S] = xi;
    p.c[S] = c;
    p.c0[S] = c;
    p.ns[S] = 0;
    float nAL, ndA, ncap;
    load_cell3(sC + c, nAL, ndA, ncap);
    put<S>(p.AL, nAL);
    put<S>(p.dA, ndA);
    put<S>(p.cap, ncap);
  }
}

__global__ void __launch_bounds__(kBlock2, 2)
mover2_kernel(const MoverArgs<float> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* sF = reinterpret_cast<double*>(smem_raw);                 // [n] fp64 accumulators
  float4* sC = reinterpret_cast<float4*>(sF + a.n_cells);           // [n] cell constants
  int32_t* sD = reinterpret_cast<int32_t*>(sC + a.n_cells);         // [n] difference array
  __shared__ int32_t s_wtot[kBlock2 / 32];

  // ---- a0: field prologue.  E^{n+1/2} = (E^n + E^{n+1})/2 (A-11), A = (q/m)E/dx on faces;
  // per cell A_L, dA = A_R - A_L (Eq. 5) and the kappa cap dtau <= sqrt(4 kappa_max/|a'|) (A-2).
  for (int c = threadIdx.x; c < a.n_cells; c += blockDim.x) {
    const int cr = (c + 1) & a.wrap_mask;
    const float AL = (float)(a.qm_over_dx * (0.5 * (a.E_n[c] + a.E_np1[c])));
    const float AR = (float)(a.qm_over_dx * (0.5 * (a.E_n[cr] + a.E_np1[cr])));
    const float dA = AR - AL;
    sC[c] = make_float4(AL, dA, a.c_cap * Prim<float>::rsqrt(fabsf(dA)), 0.0f);
    sF[c] = 0.0;
    sD[c] = 0;
  }
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1u;
  const uint32_t n32 = (uint32_t)a.n;
  uint32_t next = 0, end = 0;        // warp-uniform: the warp's current index range
  bool exhausted = false;            // the global queue has run dry
  Lane2 p;
  p.xi = p.u = p.r = p.AL = p.dA = p.cap = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    p.xa[s] = 0.0f; p.c[s] = p.c0[s] = 0; p.ns[s] = 0; p.idx[s] = 0; p.have[s] = 0;
  }
  StartAcc acc;
  acc.cell = -1; acc.f0 = acc.f1 = 0.0;
  unsigned long long tot_sub = 0;
  unsigned capped = 0;

  for (;;) {
    // A-9: an orbit that has used max_substeps with time left is parked (checked once per
    // kInner sub-steps, so it may overshoot the cap by fewer than kInner).
    if (p.ns[0] >= (uint32_t)a.max_substeps && p.r.x > 0.0f) { p.r.x = 0.0f; p.have[0] = 2; }
    if (p.ns[1] >= (uint32_t)a.max_substeps && p.r.y > 0.0f) { p.r.y = 0.0f; p.have[1] = 2; }

    // ---- a6/a7/a1: slot-level re-queue.  Parked slots wait until enough of the warp's 64 have
    // gathered, then store their results and pull the next particles of the warp's range:
    // slot 0 of the parked lanes takes the first ones, slot 1 the following ones (both runs are
    // consecutive in the binned order, so they stay coherent).
    const unsigned pk0 = __ballot_sync(kFull, !(p.r.x > 0.0f));
    const unsigned pk1 = __ballot_sync(kFull, !(p.r.y > 0.0f));
    if (pk0 | pk1) {
      const int n0 = __popc(pk0), n_parked = n0 + __popc(pk1);
      const bool go = exhausted ? (n_parked == 64) : (n_parked >= a.refill_threshold);
      if (go) {
        if (next >= end && !exhausted) {
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
        EndTerms et0, et1;
        // a lane's start-cell sums leave for the block sums when its next finished orbit began in
        // another cell: all lanes of the warp do that in the same refill, so sum them first
        warp_flush_start(sF, a.n_cells, lane, acc,
                         !(p.r.x > 0.0f) && p.have[0] && a.deposit && acc.cell >= 0 && p.c0[0] != acc.cell);
        refill_slot<0>(a, sF, sD, sC, p, acc, et0, (uint32_t)__popc(pk0 & lt_mask), next, end,
                       tot_sub, capped);
        warp_flush_start(sF, a.n_cells, lane, acc,
                         !(p.r.y > 0.0f) && p.have[1] && a.deposit && acc.cell >= 0 && p.c0[1] != acc.cell);
        refill_slot<1>(a, sF, sD, sC, p, acc, et1, (uint32_t)(n0 + __popc(pk1 & lt_mask)), next, end,
                       tot_sub, capped);
        // the two slots of a lane mostly end in the same cell: add them up first, then one
        // warp-level pass (a second one only if some lane's slots ended in different cells)
        if (et0.pending && et1.pending && et0.cell == et1.cell) {
          et0.e0 += et1.e0; et0.e1 += et1.e1; et1.pending = false;
        } else if (!et0.pending && et1.pending) {
          et0 = et1; et1.pending = false;
        }
        warp_deposit_end(sF, a.n_cells, lane, et0);
        if (__any_sync(kFull, et1.pending)) warp_deposit_end(sF, a.n_cells, lane, et1);
        next = ((uint32_t)n_parked < end - next) ? next + (uint32_t)n_parked : end;
        if (exhausted && n_parked == 64) break;
      }
    }

    // ---- kInner sub-step rounds of both slots; the warp leaves them early once no slot has an
    // orbit in flight (checked every kGroup rounds).  Sub-steps are counted per group of kGroup
    // rounds (an upper bound, for the A-9 cap and pic_stats.n_sub; exact counts: counting build).
#pragma unroll 1
    for (int j = 0; j < kInner / kGroup; ++j) {
      if (p.r.x > 0.0f) p.ns[0] += kGroup;
      if (p.r.y > 0.0f) p.ns[1] += kGroup;
#pragma unroll
      for (int g = 0; g < kGroup; ++g) substep2(a, sC, p);
      if (!__any_sync(kFull, p.r.x > 0.0f || p.r.y > 0.0f)) break;
    }
  }
  flush_start(sF, a.n_cells, acc);

  // ---- totals: warp reduce, one atomic per warp.
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tot_sub += __shfl_xor_sync(kFull, tot_sub, o);
  capped = __reduce_add_sync(kFull, capped);
  if (lane == 0) {
    atomicAdd(&a.stats[ST_SUB], tot_sub);
    if (capped) atomicAdd(&a.stats[ST_SUBSTEP_CAP], (unsigned long long)capped);
  }

  block_flush<float>(a, sF, sD, s_wtot);
}

}  // namespace picb200
