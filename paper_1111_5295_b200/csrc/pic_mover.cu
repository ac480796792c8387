// pic_mover.cu — launch side of the mover kernel (mover.cuh): launch shape, shared-memory
// budget, argument packing.  SURVEY.md 8(a) a0-a8.
#include <algorithm>
#include <cmath>

#include "mover.cuh"
#include "mover2.cuh"
#include "pic_internal.h"

// Guided self-scheduling of the work queue (mover.cuh: claim_size).  A warp claims `tile`
// (<= 512) particles while plenty are left and (what is left) / (PIC_GUIDE x warps of the grid)
// towards the end, never fewer than the minimum below: the last ranges are short, so the warps
// finish together (configs[3]: -4.7 %, configs[4] pass: -9 %, configs[2]: -0.7 %).  Species so
// small that a warp gets fewer than 192 particles in all (configs[1]) do better with one or two
// long claims per warp: every claim is a global atomic whose latency the warp waits out.
#ifndef PIC_GUIDE
#define PIC_GUIDE 4
#endif
#ifndef PIC_GUIDE_MIN
#define PIC_GUIDE_MIN 32
#endif
#ifndef PIC_GUIDE_MIN2
#define PIC_GUIDE_MIN2 64
#endif
#ifndef PIC_TINY_MIN
#define PIC_TINY_MIN 128
#endif
#ifndef PIC_TINY_MIN2
#define PIC_TINY_MIN2 256
#endif

namespace picb200 {

namespace {

// Dispatch over the kernel's template switches (CN mode, diagnostics, deposit mode, power-of-two
// grid).
template <typename T, bool P2, bool XT, typename F>
auto with_kernel_p(bool direct, bool diag, bool per_visit, F&& f) {
  const int key = (direct ? 4 : 0) | (diag ? 2 : 0) | (per_visit ? 1 : 0);
  switch (key) {
    case 0: return f(mover_kernel<T, false, false, false, P2, XT>);
    case 1: return f(mover_kernel<T, false, false, true, P2, XT>);
    case 2: return f(mover_kernel<T, false, true, false, P2, XT>);
    case 3: return f(mover_kernel<T, false, true, true, P2, XT>);
    case 4: return f(mover_kernel<T, true, false, false, P2, XT>);
    case 5: return f(mover_kernel<T, true, false, true, P2, XT>);
    case 6: return f(mover_kernel<T, true, true, false, P2, XT>);
    default: return f(mover_kernel<T, true, true, true, P2, XT>);
  }
}
// exact: the EXACT_T instantiation (fp32 only; the fp64 kernel's r is exact enough as it is)
template <typename T, typename F>
auto with_kernel(bool direct, bool diag, bool per_visit, bool pow2, bool exact, F&& f) {
  if constexpr (sizeof(T) == 4) {
    if (exact)
      return pow2 ? with_kernel_p<T, true, true>(direct, diag, per_visit, f)
                  : with_kernel_p<T, false, true>(direct, diag, per_visit, f);
  }
  return pow2 ? with_kernel_p<T, true, false>(direct, diag, per_visit, f)
              : with_kernel_p<T, false, false>(direct, diag, per_visit, f);
}

// fp32 time accounting (mover.cuh, EXACT_T): on request.
bool exact_time(const pic_params& P, double dt) {
  (void)dt;
  return (P.flags & PIC_FLAG_EXACT_TIME) != 0;
}

// GGRID instantiations (large grids): end-point deposit, generic wrap, plain time accounting.
template <typename T, typename F>
auto with_ggrid_kernel(bool direct, bool diag, F&& f) {
  const int key = (direct ? 2 : 0) | (diag ? 1 : 0);
  switch (key) {
    case 0: return f(mover_kernel<T, false, false, false, false, false, true>);
    case 1: return f(mover_kernel<T, false, true, false, false, false, true>);
    case 2: return f(mover_kernel<T, true, false, false, false, false, true>);
    default: return f(mover_kernel<T, true, true, false, false, false, true>);
  }
}

template <typename T>
cudaError_t set_smem_all(size_t bytes) {
  cudaError_t e = cudaSuccess;
  for (int key = 0; key < 32 && e == cudaSuccess; ++key)
    e = with_kernel<T>(key & 4, key & 2, key & 1, key & 8, key & 16, [&](auto k) {
      return cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    });
  return e;
}

template <typename T>
int occupancy(size_t bytes) {
  int nb = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, mover_kernel<T, true, false, false, true, false>, LaunchCfg<T>::block, bytes);
  return nb;
}

template <typename T>
void launch_t(pic_handle* h, SpeciesState& S, const double* dE_n, const double* dE_np1,
              double dt, double tol, int row0, int s) {
  const pic_params& P = h->params;
  const double dx = h->grid.length / h->grid.n_cells;
  MoverArgs<T> a;
  a.n = S.n;
  a.xi0 = (const T*)S.xi[h->cur];
  a.v0 = (const T*)S.v[h->cur];
  a.cell0 = S.cell[h->cur];
  const bool store = !(P.flags & PIC_FLAG_NO_STORE);
  a.xi1 = store ? (T*)S.xi[1 - h->cur] : nullptr;
  a.v1 = store ? (T*)S.v[1 - h->cur] : nullptr;
  a.cell1 = store ? S.cell[1 - h->cur] : nullptr;
  const bool counts = (P.flags & PIC_FLAG_COUNTS) && S.nsub;
  a.nsub_out = counts ? S.nsub : nullptr;
  a.ncross_out = counts ? S.ncross : nullptr;
  a.E_n = dE_n;
  a.E_np1 = dE_np1;
  a.n_cells = h->grid.n_cells;
  a.max_substeps = P.max_substeps;
  a.picard_max = P.picard_max;
  a.tile = S.tile;
  {
    const long long warps = (long long)S.grid_blocks * (LaunchCfg<T>::block / 32);
    a.tile_min = S.n < 192 * warps ? PIC_TINY_MIN : PIC_GUIDE_MIN;
    a.guide_div = PIC_GUIDE * (uint32_t)warps;
  }
  a.deposit = (P.flags & PIC_FLAG_NO_DEPOSIT) ? 0 : 1;
  a.wrap_mask = (h->grid.n_cells > 1 && (h->grid.n_cells & (h->grid.n_cells - 1)) == 0)
                    ? h->grid.n_cells - 1 : 0;
  // velocity-sorted warps finish in bunches: wait for a larger bunch before the refill block
  a.refill_threshold = (S.nv > 1 || S.nx > 1) ? kRefillVsort : kRefill;
  a.qm_over_dx = S.q_over_m / dx;
  a.dx = (T)dx;
  a.inv_dx = (T)(1.0 / dx);
  a.c_abs = (T)std::sqrt(2.0 * P.eps_a / dx);
  a.c_rel = (T)(2.0 * P.eps_r);
  a.c_cap = (T)std::sqrt(4.0 * P.kappa_max);
  a.dt = (T)dt;
  a.dt_exact = dt;
  // a Picard tolerance below a few ulp of the kernel precision can never be met (A-3)
  const double tol_floor = 4.0 * (sizeof(T) == 4 ? 1.1920929e-7 : 2.220446049250313e-16);
  a.tol = (T)std::max(tol, tol_floor);
  a.scale = S.w_q / dt;
  a.grid_scratch = h->d_grid_scratch;
  a.grid_stride = h->grid_stride;
  a.partial = h->d_partial + (size_t)row0 * h->grid.n_cells;
  a.queue = h->d_queue + s;
  a.stats = h->d_stats;
  const bool direct = P.cn_mode == PIC_CN_DIRECT;
  // the counting build: exact per-particle sub-step counts and anomaly counters
  const bool diag = (P.flags & (PIC_FLAG_DIAG | PIC_FLAG_COUNTS)) != 0;
  const bool per_visit = (P.flags & PIC_FLAG_DEPOSIT_PER_VISIT) != 0 && !(P.flags & PIC_FLAG_NO_DEPOSIT);
  const bool exact = sizeof(T) == 4 && exact_time(P, dt);
  if constexpr (sizeof(T) == 4) {
    // production fp32 path: two particles per lane, packed FP32 (mover2.cuh)
    if (direct && !diag && !per_visit && !exact && a.wrap_mask != 0 && S.grid_blocks2 > 0 &&
        !(P.flags & PIC_FLAG_ONE_PER_LANE)) {
      a.refill_threshold = (S.nv > 1 || S.nx > 1) ? kRefill2Vsort : kRefill2;
      a.tile = S.tile2;
      const long long warps2 = (long long)S.grid_blocks2 * (kBlock2 / 32);
      a.tile_min = S.n < 192 * warps2 ? PIC_TINY_MIN2 : PIC_GUIDE_MIN2;
      a.guide_div = PIC_GUIDE * (uint32_t)warps2;
      S.last_blocks = S.grid_blocks2;
      h->last_kernel = "mover2_kernel";
      mover2_kernel<<<dim3(S.grid_blocks2), dim3(kBlock2), h->smem_bytes2, h->stream>>>(a);
      return;
    }
  }
  S.last_blocks = S.grid_blocks;
  h->last_kernel = "mover_kernel";
  dim3 g(S.grid_blocks), b(LaunchCfg<T>::block);
  if (h->d_grid_scratch) {
    // large grid: the block's grid copy is a row of global memory (per-visit deposit and exact
    // time accounting are not instantiated for it: end-point deposit, plain accounting)
    h->last_kernel = "mover_kernel (global-memory grid)";
    with_ggrid_kernel<T>(direct, diag, [&](auto k) {
      k<<<g, b, 0, h->stream>>>(a);
      return cudaSuccess;
    });
    return;
  }
  with_kernel<T>(direct, diag, per_visit, a.wrap_mask != 0, exact, [&](auto k) {
    k<<<g, b, h->smem_bytes, h->stream>>>(a);
    return cudaSuccess;
  });
}

}  // namespace

// Shared-memory budget and launch shape.  The whole grid is staged per block (SURVEY hard part
// 6): n_cells * (8 + 4 + sizeof(T)) bytes (fp64 sums, int32 difference array, field + halo);
// B200 allows 227 KB per block.
int mover_configure(pic_handle* h) {
  const size_t bytes = h->elem == 4 ? mover_smem_bytes<float>(h->grid.n_cells)
                                    : mover_smem_bytes<double>(h->grid.n_cells);
  const bool ggrid = bytes > 220 * 1024;       // the grid does not fit a block's shared memory
  h->smem_bytes = ggrid ? 0 : bytes;
  int occ;
  if (ggrid) {
    if (h->params.flags & PIC_FLAG_DEPOSIT_PER_VISIT)
      return set_err(h, PIC_ERR_UNSUPPORTED, "per-visit deposit needs the grid in shared memory (n_cells too large)");
    if ((h->params.flags & PIC_FLAG_EXACT_TIME) && h->elem == 4)
      return set_err(h, PIC_ERR_UNSUPPORTED, "exact time accounting is not built for grids beyond shared memory (n_cells too large)");
    h->grid_stride = (bytes + 255) & ~(size_t)255;
    // one wave of blocks, but no more rows of scratch than ~2 GB
    const size_t budget = (size_t)2 << 30;
    occ = (int)std::max<size_t>(1, std::min<size_t>(2, budget / h->grid_stride / h->sm_count));
    h->ggrid_max_blocks = (int)std::max<size_t>(1, std::min<size_t>((size_t)h->sm_count * occ, budget / h->grid_stride));
  } else {
    cudaError_t e = h->elem == 4 ? set_smem_all<float>(bytes) : set_smem_all<double>(bytes);
    if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "cudaFuncSetAttribute(smem)", e);
    occ = h->elem == 4 ? occupancy<float>(bytes) : occupancy<double>(bytes);
    if (occ < 1) return set_err(h, PIC_ERR_CUDA, "mover kernel does not fit on an SM");
  }
  h->blocks_per_sm = occ;
  int rows = 0;
  for (auto& S : h->sp) {
    // persistent grid: one wave of resident blocks (a multiple of the SM count), fewer for
    // small problems so that every warp still gets a few refills' worth of particles.
    const long long full = ggrid ? h->ggrid_max_blocks : (long long)h->sm_count * occ;
    const int block = h->elem == 4 ? LaunchCfg<float>::block : LaunchCfg<double>::block;
    const long long want = (S.n + block * 4 - 1) / (block * 4);
    S.grid_blocks = (int)std::max<long long>(1, std::min(full, want));
    const long long warps = (long long)S.grid_blocks * (block / 32);
    long long tile = S.n / (warps * 8);                 // >= 8 claims per warp
#ifndef PIC_TILE_MIN
#define PIC_TILE_MIN 128
#endif
#ifndef PIC_TILE_MIN2
#define PIC_TILE_MIN2 256
#endif
#ifndef PIC_TILE_MAX
#define PIC_TILE_MAX 512
#endif
    tile = std::max<long long>(PIC_TILE_MIN, std::min<long long>(PIC_TILE_MAX, tile / 32 * 32));
    S.tile = (int)tile;
    rows += S.grid_blocks;
  }
  // two-per-lane fp32 kernel: power-of-two grids whose 28 B per cell leave two blocks per SM
  const int32_t ng = h->grid.n_cells;
  if (h->elem == 4 && ng > 1 && (ng & (ng - 1)) == 0) {
    const size_t b2 = mover2_smem_bytes(ng);
    int occ2 = 0;
    if (b2 <= 113 * 1024 &&
        cudaFuncSetAttribute(mover2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)b2) == cudaSuccess &&
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, mover2_kernel, kBlock2, b2) == cudaSuccess &&
        occ2 >= 2) {
      h->smem_bytes2 = b2;
      for (auto& S : h->sp) {
        const long long full = (long long)h->sm_count * occ2;
        const long long want = (S.n + kBlock2 * 8 - 1) / (kBlock2 * 8);
        S.grid_blocks2 = (int)std::max<long long>(1, std::min<long long>(std::min(full, want), S.grid_blocks));
        const long long warps = (long long)S.grid_blocks2 * (kBlock2 / 32);
        long long tile = S.n / (warps * 8);
        tile = std::max<long long>(PIC_TILE_MIN2, std::min<long long>(PIC_TILE_MAX, tile / 64 * 64));
        S.tile2 = (int)tile;
      }
    } else {
      cudaGetLastError();
    }
  }
  h->total_rows = rows;
  if (ggrid) {
    int maxb = 1;
    for (auto& S : h->sp) maxb = std::max(maxb, S.grid_blocks);
    cudaError_t e = cudaMalloc(&h->d_grid_scratch, h->grid_stride * (size_t)maxb);
    if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "cudaMalloc(global-memory grid)", e);
  }
  return PIC_OK;
}

int launch_mover(pic_handle* h, int s, const double* dE_n, const double* dE_np1, double dt,
                 double tol, int row0) {
  SpeciesState& S = h->sp[s];
  if (h->elem == 4) launch_t<float>(h, S, dE_n, dE_np1, dt, tol, row0, s);
  else launch_t<double>(h, S, dE_n, dE_np1, dt, tol, row0, s);
  h->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "mover_kernel launch", e);
  return PIC_OK;
}

}  // namespace picb200
