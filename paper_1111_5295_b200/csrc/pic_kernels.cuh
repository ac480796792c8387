// pic_kernels.cuh — small device kernels around the mover: binning by cell,
// block-partial reduction (a8), Ampere residual (a9), diagnostics.  None of these is the hot loop.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pic_check.cuh"

namespace picb200 {

// Sort key of the binning: cell only (nx = nv = 1), or with PIC_FLAG_VSORT the phase-space cell
// (cell, xi class, velocity class) -- the paper's phase-space sort: nx classes of
// the in-cell offset and nv velocity classes over [vmean - 4 sigma, vmean + 4 sigma], ordered so
// that neighbours in memory share the cell and the offset class and have adjacent velocities.
// Lanes of a warp then start almost the same orbit: same sub-step sequence, crossings in the same
// round, orbit ends in the same round.
//
// PIC_FLAG_STRIDED orders the same three sub-keys the other way round, (velocity class, offset
// class, cell): the paper's own layout (Eq. 15), in which consecutive threads hold
// particles of CONSECUTIVE cells with similar velocities (made for its per-warp atomic deposits,
// where lanes sharing a cell collide).  With about one particle per key the offset class plays
// the part of the paper's index p of a particle inside its phase-space cell.  Kept for the A/B
// of SURVEY 8(f) #3 (profiles/r2_strided_layout.md).
struct VKey {
  int32_t nx, nv;
  double vmean, vinv;   // vinv = nv / (8 sigma)
  int32_t n_cells;      // number of cells
  int32_t strided;      // != 0: strided order (v class, offset class, cell); 0: cell-major order
};
__device__ __forceinline__ int32_t sort_key(const VKey& k, int32_t cell, double xi, double v) {
  cell = chk(cell, k.n_cells);
  if (k.nv <= 1 && k.nx <= 1) return cell;
  const double t = (v - k.vmean) * k.vinv + 0.5 * k.nv;
  const int32_t b = (int32_t)fmin(fmax(t, 0.0), (double)(k.nv - 1));
  const int32_t xb = min((int32_t)(xi * k.nx), k.nx - 1);
  const int32_t key = k.strided ? (b * k.nx + xb) * k.n_cells + cell : (cell * k.nx + xb) * k.nv + b;
  return chk(key, (long long)k.n_cells * k.nx * k.nv);
}

// sum v, sum v^2 (fp64) -> out[0], out[1]
static __global__ void moments_kernel(long long n, const double* __restrict__ v, double* __restrict__ out) {
  __shared__ double r0[32], r1[32];
  double s = 0.0, q = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const double t = v[i];
    s += t; q += t * t;
  }
  for (int o = 16; o > 0; o >>= 1) {
    s += __shfl_xor_sync(0xffffffffu, s, o);
    q += __shfl_xor_sync(0xffffffffu, q, o);
  }
  if ((threadIdx.x & 31) == 0) { r0[threadIdx.x >> 5] = s; r1[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { a += r0[w]; b += r1[w]; }
    atomicAdd(&out[0], a);
    atomicAdd(&out[1], b);
  }
}

// x -> (cell, xi): cell = floor(x/dx) clipped to [0, n_cells-1], xi = x/dx - cell clipped to
// [0,1] and rounded to T.  Also the per-cell histogram and input validation (flag != 0 if any
// x is outside [0,L) or x / v is not finite).
template <typename T>
__global__ void bin_kernel(long long n, const double* __restrict__ x, const double* __restrict__ v,
                           double dx, double length, int32_t n_cells, int32_t* __restrict__ cell,
                           T* __restrict__ xi, T* __restrict__ vout, int32_t* __restrict__ hist,
                           int32_t* __restrict__ flag, VKey vk) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const double xv = x[i], vv = v[i];
    if (!(xv >= 0.0 && xv < length) || !isfinite(vv)) { atomicOr(flag, 1); }
    const double u = xv / dx;
    double fc = floor(u);
    if (!(fc >= 0.0)) fc = 0.0;
    if (fc > (double)(n_cells - 1)) fc = (double)(n_cells - 1);
    const int32_t c = (int32_t)fc;
    double o = u - fc;
    o = o < 0.0 ? 0.0 : (o > 1.0 ? 1.0 : o);
    cell[i] = c;
    xi[i] = (T)o;
    vout[i] = (T)vv;
    atomicAdd(&hist[sort_key(vk, c, (double)(T)o, (double)(T)vv)], 1);
  }
}

template <typename T>
__global__ void hist_kernel(long long n, const int32_t* __restrict__ cell, const T* __restrict__ xi,
                            const T* __restrict__ v, int32_t* __restrict__ hist, VKey vk) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x)
    atomicAdd(&hist[sort_key(vk, cell[i], (double)xi[i], (double)v[i])], 1);
}

// Exclusive scan of hist[0..n) in place, three passes: per-chunk sums, scan of the chunk sums
// (one block), per-chunk exclusive scan + offset.  kScanChunk elements per block.
constexpr int kScanChunk = 4096;
constexpr int kScanThreads = 512;

static __device__ __forceinline__ int32_t block_exclusive_scan(int32_t val, int32_t* wsum, int32_t& total) {
  // exclusive scan of one value per thread over a kScanThreads block
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int32_t inc = val;
  for (int o = 1; o < 32; o <<= 1) {
    const int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    int32_t s = lane < (int)(blockDim.x >> 5) ? wsum[lane] : 0;
    for (int o = 1; o < 32; o <<= 1) {
      const int32_t t = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += t;
    }
    wsum[lane] = s;   // inclusive over warps
  }
  __syncthreads();
  total = wsum[(blockDim.x >> 5) - 1];
  const int32_t r = (w ? wsum[w - 1] : 0) + inc - val;
  __syncthreads();
  return r;
}

static __global__ void scan_sums_kernel(long long n, const int32_t* __restrict__ hist,
                                        int32_t* __restrict__ sums) {
  __shared__ int32_t red[32];
  const long long base = (long long)blockIdx.x * kScanChunk;
  int32_t s = 0;
  for (int i = threadIdx.x; i < kScanChunk; i += blockDim.x)
    if (base + i < n) s += hist[base + i];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    int32_t t = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
    sums[blockIdx.x] = t;
  }
}

// one block: exclusive scan of sums[0..m) in place (m = number of chunks, any size)
static __global__ void scan_top_kernel(int32_t m, int32_t* __restrict__ sums) {
  __shared__ int32_t wsum[32];
  __shared__ int32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < m; base += blockDim.x) {
    const int i = base + threadIdx.x;
    const int32_t val = i < m ? sums[i] : 0;
    int32_t total;
    const int32_t ex = block_exclusive_scan(val, wsum, total);
    if (i < m) sums[i] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry += total;
    __syncthreads();
  }
}

static __global__ void scan_chunks_kernel(long long n, int32_t* __restrict__ hist,
                                          const int32_t* __restrict__ sums) {
  __shared__ int32_t wsum[32];
  constexpr int per = kScanChunk / kScanThreads;
  const long long base = (long long)blockIdx.x * kScanChunk + (long long)threadIdx.x * per;
  int32_t v[per];
  int32_t s = 0;
#pragma unroll
  for (int j = 0; j < per; ++j) {
    v[j] = (base + j < n) ? hist[base + j] : 0;
    s += v[j];
  }
  int32_t total;
  int32_t run = sums[blockIdx.x] + block_exclusive_scan(s, wsum, total);
#pragma unroll
  for (int j = 0; j < per; ++j) {
    if (base + j < n) hist[base + j] = run;
    run += v[j];
  }
}

// Scatter into cell bins.  hist holds the running cursor of each cell (exclusive scan at entry).
// Order inside a bin is arbitrary; `id` carries the original index.
template <typename T>
__global__ void scatter_kernel(long long n, const int32_t* __restrict__ cell_in,
                               const T* __restrict__ xi_in, const T* __restrict__ v_in,
                               const uint32_t* __restrict__ id_in, int32_t* __restrict__ cursor,
                               int32_t* __restrict__ cell_out, T* __restrict__ xi_out,
                               T* __restrict__ v_out, uint32_t* __restrict__ id_out, VKey vk) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const int32_t c = cell_in[i];
    const int32_t dst =
        chk(atomicAdd(&cursor[sort_key(vk, c, (double)xi_in[i], (double)v_in[i])], 1), n);
    cell_out[dst] = c;
    xi_out[dst] = xi_in[i];
    v_out[dst] = v_in[i];
    id_out[dst] = id_in ? id_in[i] : (uint32_t)i;
  }
}

// a8: jbar_f = sum over block rows (fixed order -> reproducible given the rows).  A block of
// kRedCols x kRedRows threads owns kRedCols faces: thread (c, r) adds rows r, r + kRedRows, ...
// of its face (coalesced across c), then the kRedRows partial sums are added in order.  (One
// thread per face looping over all rows was latency-bound: 64 us for 592 rows x 512 faces.)
constexpr int kRedCols = 32, kRedRows = 16;
static __global__ void __launch_bounds__(kRedCols * kRedRows)
reduce_rows_kernel(int rows, int32_t n_cells, const double* __restrict__ partial,
                   double* __restrict__ jbar) {
  __shared__ double sm[kRedRows][kRedCols + 1];
  const int c = threadIdx.x, r0 = threadIdx.y;
  const int f = blockIdx.x * kRedCols + c;
  double s = 0.0;
  if (f < n_cells)
    for (int r = r0; r < rows; r += kRedRows) s += partial[(size_t)r * n_cells + f];
  sm[r0][c] = s;
  __syncthreads();
  if (r0 == 0 && f < n_cells) {
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < kRedRows; ++k) t += sm[k][c];
    jbar[f] = t;
  }
}

// a9: R_f = (E^{n+1}_f - E^n_f)/dt + jbar_f - <jbar>  (eps0 = 1).  One block.
// resid[n_cells] receives the number of orbits cut off at max_substeps (A-9), so that one copy
// brings both back.
static __global__ void residual_kernel(int32_t n_cells, const double* __restrict__ E_n,
                                const double* __restrict__ E_np1, double dt,
                                const double* __restrict__ jbar, double* __restrict__ resid,
                                const unsigned long long* __restrict__ n_capped) {
  __shared__ double red[32];
  __shared__ double mean;
  double s = 0.0;
  for (int f = threadIdx.x; f < n_cells; f += blockDim.x) s += jbar[f];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
    mean = t / n_cells;
  }
  __syncthreads();
  for (int f = threadIdx.x; f < n_cells; f += blockDim.x)
    resid[f] = (E_np1[f] - E_n[f]) / dt + jbar[f] - mean;
  if (threadIdx.x == 0) resid[n_cells] = (double)*n_capped;
}

// Getter: un-permute to the original order.  Any output may be NULL.
template <typename T>
__global__ void unpermute_kernel(long long n, const uint32_t* __restrict__ id,
                                 const T* __restrict__ xi, const T* __restrict__ v,
                                 const int32_t* __restrict__ cell, double dx, double* x_out,
                                 double* v_out, int32_t* cell_out, double* xi_out) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const uint32_t j = chk(id[i], n);
    const double o = (double)xi[i];
    const int32_t c = cell[i];
    if (x_out) x_out[j] = ((double)c + o) * dx;
    if (v_out) v_out[j] = (double)v[i];
    if (cell_out) cell_out[j] = c;
    if (xi_out) xi_out[j] = o;
  }
}

static __global__ void unpermute_counts_kernel(long long n, const uint32_t* __restrict__ id,
                                        const uint32_t* __restrict__ a, const uint32_t* __restrict__ b,
                                        uint32_t* a_out, uint32_t* b_out) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const uint32_t j = chk(id[i], n);
    if (a_out) a_out[j] = a[i];
    if (b_out) b_out[j] = b[i];
  }
}

// pic_copy_state: element-wise conversion between the precisions of two handles.
template <typename TS, typename TD>
__global__ void convert_kernel(long long n, const TS* __restrict__ a, TD* __restrict__ b) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x)
    b[i] = (TD)a[i];
}

// sum_p v_p^2 (fp64), one atomic per block.
template <typename T>
__global__ void sumsq_kernel(long long n, const T* __restrict__ v, double* __restrict__ out) {
  __shared__ double red[32];
  double s = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const double t = (double)v[i];
    s += t * t;
  }
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
    atomicAdd(out, t);
  }
}

// rho on cell centres, quadratic B-spline (A-10): with p = xi in [0,1] inside cell c the
// weights on cells c-1, c, c+1 are (1-p)^2/2, 3/4 - (p-1/2)^2, p^2/2.  The state is binned by
// cell, so every thread takes kRhoChunk CONSECUTIVE particles and keeps the three sums of the
// current cell in registers; they go to memory when the cell changes and at the end of the
// chunk, there summed over the warp first when all its lanes are in the same cell, into the
// block's shared-memory copy of rho (global fp64 atomics per particle took 1.1 ms at 2e6
// particles).
constexpr int kRhoChunk = 32;
__device__ __forceinline__ void rho_flush(double* __restrict__ rho, int32_t n_cells, int32_t c,
                                          double wl, double wc, double wr) {
  c = chk(c, n_cells);
  atomicAdd(&rho[c == 0 ? n_cells - 1 : c - 1], wl);
  atomicAdd(&rho[c], wc);
  atomicAdd(&rho[c + 1 == n_cells ? 0 : c + 1], wr);
}
// Persistent blocks: each owns one contiguous span of the particle list and a shared-memory copy
// of rho (dynamic, n_cells doubles), flushed to global memory once at the end.
// SMEM = false (grids too large for shared memory): the sums go straight to global memory.
template <typename T, bool SMEM = true>
__global__ void rho_kernel(long long n, const T* __restrict__ xi, const int32_t* __restrict__ cell,
                           int32_t n_cells, double w_over_dx, double* __restrict__ rho) {
  extern __shared__ double s_rho_dyn[];
  double* s_rho = SMEM ? s_rho_dyn : rho;
  if (SMEM) {
    for (int f = threadIdx.x; f < n_cells; f += blockDim.x) s_rho[f] = 0.0;
    __syncthreads();
  }
  const long long stride = (long long)blockDim.x * kRhoChunk;
  const long long per_block = ((n + gridDim.x - 1) / gridDim.x + stride - 1) / stride * stride;
  const long long b0 = blockIdx.x * per_block;
  const long long b1 = b0 + per_block < n ? b0 + per_block : n;
  const unsigned full = 0xffffffffu;
  // the trip count is the same for every thread of the block (a lane past the end has an empty run)
  for (long long base = b0; base < b1; base += stride) {
    const long long i0 = base + (long long)threadIdx.x * kRhoChunk;
    const long long i1 = i0 + kRhoChunk < b1 ? i0 + kRhoChunk : b1;
    int32_t cur = -1;
    double wl = 0.0, wc = 0.0, wr = 0.0;
    for (long long i = i0; i < i1; ++i) {
      const int32_t c = cell[i];
      if (c != cur) {
        if (cur >= 0) rho_flush(s_rho, n_cells, cur, wl, wc, wr);
        cur = c;
        wl = wc = wr = 0.0;
      }
      const double p = (double)xi[i];
      wl += w_over_dx * 0.5 * (1.0 - p) * (1.0 - p);
      wc += w_over_dx * (0.75 - (p - 0.5) * (p - 0.5));
      wr += w_over_dx * 0.5 * p * p;
    }
    const int32_t c0 = __shfl_sync(full, cur, 0);
    if (__all_sync(full, cur == c0 && cur >= 0)) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        wl += __shfl_xor_sync(full, wl, o);
        wc += __shfl_xor_sync(full, wc, o);
        wr += __shfl_xor_sync(full, wr, o);
      }
      if ((threadIdx.x & 31) == 0) rho_flush(s_rho, n_cells, cur, wl, wc, wr);
    } else if (cur >= 0) {
      rho_flush(s_rho, n_cells, cur, wl, wc, wr);
    }
  }
  if (SMEM) {
    __syncthreads();
    for (int f = threadIdx.x; f < n_cells; f += blockDim.x)
      if (s_rho[f] != 0.0) atomicAdd(&rho[f], s_rho[f]);
  }
}

// Histogram of per-particle counts (BJ configs[3]: sub-step histogram): bin k holds the particles
// with k*width <= v < (k+1)*width, the last bin everything above.  Per-block shared-memory
// histogram (native 32-bit ATOMS), one global 64-bit add per non-empty bin and block.
constexpr int kHistMaxBins = 4096;
static __global__ void count_hist_kernel(long long n, const uint32_t* __restrict__ v, uint32_t width,
                                         int n_bins, unsigned long long* __restrict__ out) {
  extern __shared__ uint32_t s_h[];
  for (int b = threadIdx.x; b < n_bins; b += blockDim.x) s_h[b] = 0;
  __syncthreads();
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const uint32_t b = v[i] / width;
    atomicAdd(&s_h[b < (uint32_t)n_bins ? b : (uint32_t)n_bins - 1u], 1u);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < n_bins; b += blockDim.x)
    if (s_h[b]) atomicAdd(&out[b], (unsigned long long)s_h[b]);
}

}  // namespace picb200
