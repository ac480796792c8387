// pic_api.cu — the C-ABI of include/pic.h: handle life cycle, binning, move, residual, commit,
// getters.  Argument marshalling and launches only; the arithmetic of the path is in mover.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "mover.cuh"
#include "pic_internal.h"
#include "pic_kernels.cuh"

namespace picb200 {

#if PIC_BOUNDS_CHECK
__device__ unsigned long long g_bounds_violations = 0;   // pic_check.cuh
namespace {
__global__ void bounds_self_test_kernel(int* sink) { sink[chk(5, 3)] = 1; }   // one violation
}  // namespace
#endif

int set_err(pic_handle* h, int code, const char* what, cudaError_t ce) {
  if (h) {
    h->err = what ? what : "";
    if (ce != cudaSuccess) {
      h->err += ": ";
      h->err += cudaGetErrorString(ce);
    }
  }
  return code;
}

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

namespace {

int grid_for(long long n, int threads = 256, int cap = 148 * 16) {
  long long g = (n + threads - 1) / threads;
  return (int)std::max<long long>(1, std::min<long long>(g, cap));
}

// Bring a caller grid array to the device (no-op for device pointers).
int to_device(pic_handle* h, const double* src, double* staging, const double** out) {
  if (is_device_ptr(src)) { *out = src; return PIC_OK; }
  PIC_CUDA(h, cudaMemcpyAsync(staging, src, sizeof(double) * h->grid.n_cells,
                              cudaMemcpyHostToDevice, h->stream));
  *out = staging;
  return PIC_OK;
}

// Deliver a device grid array to the caller (host: copy + synchronise).
int from_device(pic_handle* h, const double* dsrc, double* dst) {
  if (!dst) return PIC_OK;
  const bool dev = is_device_ptr(dst);
  PIC_CUDA(h, cudaMemcpyAsync(dst, dsrc, sizeof(double) * h->grid.n_cells,
                              dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  if (!dev) PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  return PIC_OK;
}

VKey key_of(const pic_handle* h, const SpeciesState& S) {
  return VKey{S.nx, S.nv, S.vmean, S.vinv, h->grid.n_cells, S.strided ? 1 : 0};
}

// exclusive scan of d_hist[0..nk) (three small kernels)
int scan_hist(pic_handle* h, long long nk) {
  const int chunks = (int)((nk + kScanChunk - 1) / kScanChunk);
  scan_sums_kernel<<<chunks, kScanThreads, 0, h->stream>>>(nk, h->d_hist, h->d_scan);
  scan_top_kernel<<<1, kScanThreads, 0, h->stream>>>(chunks, h->d_scan);
  scan_chunks_kernel<<<chunks, kScanThreads, 0, h->stream>>>(nk, h->d_hist, h->d_scan);
  h->launches += 3;
  PIC_CUDA(h, cudaGetLastError());
  return PIC_OK;
}

template <typename T>
int bin_species(pic_handle* h, SpeciesState& S, const double* dx_, const double* dv_) {
  const int32_t ng = h->grid.n_cells;
  const double dx = h->grid.length / ng;
  const int b = h->cur;
  S.nx = 1;
  S.nv = 1;
  if (h->params.flags & PIC_FLAG_VSORT) {
    // velocity classes: mean and sigma of the species' velocities (fp64 reduction, init only)
    double* dm = nullptr;
    double hm[2] = {0.0, 0.0};
    PIC_CUDA(h, cudaMalloc(&dm, 2 * sizeof(double)));
    cudaMemsetAsync(dm, 0, 2 * sizeof(double), h->stream);
    moments_kernel<<<grid_for(S.n), 256, 0, h->stream>>>(S.n, dv_, dm);
    cudaError_t e = cudaMemcpyAsync(hm, dm, sizeof hm, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(dm);
    h->launches++;
    if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "velocity moments", e);
    const double mean = hm[0] / (double)S.n;
    const double var = hm[1] / (double)S.n - mean * mean;
    // classes: about 4 particles per phase-space cell, nx = 8 (or 4) offset classes, nv <= 1024
    // velocity classes (powers of two), at most n_keys keys in all
    const double ppc = (double)S.n / ng;
#ifndef PIC_NX
#define PIC_NX 8
#endif
#ifndef PIC_NX2
#define PIC_NX2 4
#endif
#ifndef PIC_PPK
#define PIC_PPK 4
#endif
    // offset classes: 8 for the one-particle-per-lane kernels; the two-per-lane fp32 kernel
    // (64 orbits per warp) does better with 4 and twice as fine velocity classes
    // (profiles/r2_bench.md)
    const bool pow2 = ng > 1 && (ng & (ng - 1)) == 0;
    const bool two_per_lane = h->elem == 4 && pow2 && h->params.cn_mode == PIC_CN_DIRECT &&
        (size_t)ng * 28 <= 113 * 1024 &&
        !(h->params.flags & (PIC_FLAG_ONE_PER_LANE | PIC_FLAG_DEPOSIT_PER_VISIT));
    int32_t nx = two_per_lane ? PIC_NX2 : PIC_NX, nv = 1;
#ifndef PIC_NVMAX
#define PIC_NVMAX 1024
#endif
    const bool strided = (h->params.flags & PIC_FLAG_STRIDED) != 0;
    if (strided) {
      // about one particle per key: 256 velocity rows (fewer for thin species), the rest of the
      // particles of a cell spread over offset classes
#ifndef PIC_STRIDE_NV
#define PIC_STRIDE_NV 256
#endif
#ifndef PIC_STRIDE_PPK
#define PIC_STRIDE_PPK 1
#endif
      nx = 1;
      while (nv < PIC_STRIDE_NV && (double)nv * 2 * 2 <= ppc) nv *= 2;
      while (nx < 4096 && (double)nx * 2 * nv * PIC_STRIDE_PPK <= ppc) nx *= 2;
    } else
    while (nv < PIC_NVMAX && (double)nx * nv * 2 * PIC_PPK <= ppc) nv *= 2;
    while (nx > 1 && (long long)ng * nx * nv > h->n_keys) nx /= 2;
    while (nv > 1 && (long long)ng * nx * nv > h->n_keys) nv /= 2;
    if (var > 0.0 && nv > 1) {
      S.nx = nx;
      S.nv = nv;
      S.vmean = mean;
      S.vinv = (double)nv / (8.0 * std::sqrt(var));
      S.strided = strided;
    }
  }
  const VKey vk = key_of(h, S);
  const long long nk = (long long)ng * S.nx * S.nv;
  // stage 1: cell/xi/v in input order into buffer 1-b, histogram over the sort keys
  PIC_CUDA(h, cudaMemsetAsync(h->d_hist, 0, sizeof(int32_t) * (nk + 1), h->stream));
  bin_kernel<T><<<grid_for(S.n), 256, 0, h->stream>>>(S.n, dx_, dv_, dx, h->grid.length, ng,
                                                      S.cell[1 - b], (T*)S.xi[1 - b],
                                                      (T*)S.v[1 - b], h->d_hist, h->d_flag, vk);
  if (int rc = scan_hist(h, nk)) return rc;
  scatter_kernel<T><<<grid_for(S.n), 256, 0, h->stream>>>(
      S.n, S.cell[1 - b], (const T*)S.xi[1 - b], (const T*)S.v[1 - b], nullptr, h->d_hist,
      S.cell[b], (T*)S.xi[b], (T*)S.v[b], S.id[b], vk);
  h->launches += 2;
  PIC_CUDA(h, cudaGetLastError());
  return PIC_OK;
}

template <typename T>
int rebin_species(pic_handle* h, SpeciesState& S) {
  // state n+1 lives in buffer 1-cur; scatter it, binned, into buffer cur (old state n is dead).
  const int32_t ng = h->grid.n_cells;
  const int src = 1 - h->cur, dst = h->cur;
  const VKey vk = key_of(h, S);
  const long long nk = (long long)ng * S.nx * S.nv;
  if (nk > h->n_keys) return set_err(h, PIC_ERR_STATE, "rebin: sort key larger than the binning scratch");
  PIC_CUDA(h, cudaMemsetAsync(h->d_hist, 0, sizeof(int32_t) * (nk + 1), h->stream));
  hist_kernel<T><<<grid_for(S.n), 256, 0, h->stream>>>(S.n, S.cell[src], (const T*)S.xi[src],
                                                       (const T*)S.v[src], h->d_hist, vk);
  if (int rc = scan_hist(h, nk)) return rc;
  // ids: buffer 1-cur was written in the order of buffer cur, so its ids are id[cur]; the
  // re-binned ids go to id[1-cur] and the two id arrays then trade places.
  scatter_kernel<T><<<grid_for(S.n), 256, 0, h->stream>>>(
      S.n, S.cell[src], (const T*)S.xi[src], (const T*)S.v[src], S.id[dst], h->d_hist,
      S.cell[dst], (T*)S.xi[dst], (T*)S.v[dst], S.id[src], vk);
  std::swap(S.id[0], S.id[1]);
  h->launches += 2;
  PIC_CUDA(h, cudaGetLastError());
  return PIC_OK;
}

void free_all(pic_handle* h) {
  for (auto& S : h->sp) {
    for (int b = 0; b < 2; ++b) {
      cudaFree(S.xi[b]); cudaFree(S.v[b]); cudaFree(S.cell[b]); cudaFree(S.id[b]);
    }
    cudaFree(S.nsub); cudaFree(S.ncross);
  }
  cudaFree(h->dE_n); cudaFree(h->dE_step); cudaFree(h->dE_np1); cudaFree(h->d_jbar);
  cudaFree(h->d_resid); cudaFree(h->d_partial); cudaFree(h->d_queue);   // d_stats is part of d_queue
  cudaFree(h->d_hist); cudaFree(h->d_flag); cudaFree(h->d_scan); cudaFree(h->d_grid_scratch);
  if (h->h_pin) cudaFreeHost(h->h_pin);
  for (auto& e : h->graphs) cudaGraphExecDestroy(e.exec);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  if (h->ev_pin) cudaEventDestroy(h->ev_pin);
}

thread_local std::string g_init_err;

}  // namespace
}  // namespace picb200

using namespace picb200;

namespace {
template <typename TS, typename TD>
void convert_arr(pic_handle* d, long long n, const void* a, void* b) {
  picb200::convert_kernel<TS, TD><<<grid_for(n), 256, 0, d->stream>>>(n, (const TS*)a, (TD*)b);
  d->launches++;
}
}  // namespace

extern "C" {

int pic_init(pic_handle** out, const pic_grid* grid, const pic_species* species, int n_species,
             const double* const* x, const double* const* v, const pic_params* params,
             void* stream) {
  if (!out) return PIC_ERR_ARG;
  *out = nullptr;
  if (!grid || !species || !x || !v || !params || n_species < 1 || grid->n_cells < 1 ||
      !(grid->length > 0.0) || !(params->eps_a > 0.0) || !(params->eps_r > 0.0) ||
      !(params->kappa_max > 0.0 && params->kappa_max < 1.0) || params->max_substeps < 1 ||
      (params->precision != PIC_FP32 && params->precision != PIC_FP64) ||
      (params->cn_mode != PIC_CN_PICARD && params->cn_mode != PIC_CN_DIRECT))
    return PIC_ERR_ARG;
  for (int s = 0; s < n_species; ++s)
    if (species[s].n < 0 || species[s].n > 0x7fffffffLL || !x[s] || !v[s] ||
        species[s].q_over_m == 0.0)
      return PIC_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return PIC_ERR_CUDA;   // no CPU fallback
  }
  pic_handle* h = new (std::nothrow) pic_handle();
  if (!h) return PIC_ERR_ARG;
  h->grid = *grid;
  h->params = *params;
  if (h->params.picard_max < 1) h->params.picard_max = 100;
  h->stream = (cudaStream_t)stream;
  h->elem = params->precision == PIC_FP32 ? 4 : 8;
  int rc = PIC_OK;
  auto fail = [&](int code) { free_all(h); g_init_err = h->err; delete h; return code; };
  {
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
      return fail(set_err(h, PIC_ERR_CUDA, "cudaGetDeviceProperties"));
    h->sm_count = prop.multiProcessorCount;
  }
  const int32_t ng = grid->n_cells;
#define INIT_CUDA(call)                                                                    \
  do {                                                                                     \
    cudaError_t ce_ = (call);                                                              \
    if (ce_ != cudaSuccess) return fail(set_err(h, PIC_ERR_CUDA, #call, ce_));             \
  } while (0)
  INIT_CUDA(cudaMalloc(&h->dE_n, sizeof(double) * ng));
  INIT_CUDA(cudaMalloc(&h->dE_step, sizeof(double) * ng));
  INIT_CUDA(cudaMalloc(&h->dE_np1, sizeof(double) * ng));
  INIT_CUDA(cudaMalloc(&h->d_jbar, sizeof(double) * ng));
  INIT_CUDA(cudaMalloc(&h->d_resid, sizeof(double) * (ng + 1)));   // + the sub-step-cap count
  // queue counters and stats in one allocation: one memset per move
  INIT_CUDA(cudaMalloc(&h->d_queue, sizeof(unsigned long long) * (n_species + ST_COUNT)));
  h->d_stats = h->d_queue + n_species;
  INIT_CUDA(cudaMallocHost(&h->h_pin, sizeof(double) * 2 * (ng + 1)));   // staging of E in / R out
#ifndef PIC_KEYCAP_LOG2
#define PIC_KEYCAP_LOG2 24
#endif
  // sort keys: cells x offset classes x velocity classes, at most 2^24 keys (64 MB of counters)
  h->n_keys = (params->flags & PIC_FLAG_VSORT)
                  ? std::max<long long>(ng, std::min<long long>((long long)ng * 65536, 1LL << PIC_KEYCAP_LOG2))
                  : ng;
  INIT_CUDA(cudaMalloc(&h->d_hist, sizeof(int32_t) * (h->n_keys + 1)));
  INIT_CUDA(cudaMalloc(&h->d_scan, sizeof(int32_t) * (h->n_keys / kScanChunk + 2)));
  INIT_CUDA(cudaMalloc(&h->d_flag, sizeof(int32_t)));
  INIT_CUDA(cudaMemsetAsync(h->d_flag, 0, sizeof(int32_t), h->stream));
  INIT_CUDA(cudaEventCreate(&h->ev0));
  INIT_CUDA(cudaEventCreate(&h->ev1));
  INIT_CUDA(cudaEventCreateWithFlags(&h->ev_pin, cudaEventDisableTiming));
  h->sp.resize(n_species);
  for (int s = 0; s < n_species; ++s) {
    SpeciesState& S = h->sp[s];
    S.n = species[s].n;
    S.q_over_m = species[s].q_over_m;
    S.w_q = species[s].macro_charge;
    const size_t n1 = (size_t)std::max<long long>(S.n, 1);
    for (int b = 0; b < 2; ++b) {
      INIT_CUDA(cudaMalloc(&S.xi[b], h->elem * n1));
      INIT_CUDA(cudaMalloc(&S.v[b], h->elem * n1));
      INIT_CUDA(cudaMalloc(&S.cell[b], sizeof(int32_t) * n1));
      INIT_CUDA(cudaMalloc(&S.id[b], sizeof(uint32_t) * n1));
    }
    if (params->flags & PIC_FLAG_COUNTS) {
      INIT_CUDA(cudaMalloc(&S.nsub, sizeof(uint32_t) * n1));
      INIT_CUDA(cudaMalloc(&S.ncross, sizeof(uint32_t) * n1));
    }
    if (S.n == 0) continue;
    // inputs: device pointers are used in place, host arrays go through a temporary
    const double* dxp = x[s];
    const double* dvp = v[s];
    double *tx = nullptr, *tv = nullptr;
    if (!is_device_ptr(x[s])) {
      INIT_CUDA(cudaMalloc(&tx, sizeof(double) * S.n));
      INIT_CUDA(cudaMemcpyAsync(tx, x[s], sizeof(double) * S.n, cudaMemcpyHostToDevice, h->stream));
      dxp = tx;
    }
    if (!is_device_ptr(v[s])) {
      cudaError_t e = cudaMalloc(&tv, sizeof(double) * S.n);
      if (e == cudaSuccess)
        e = cudaMemcpyAsync(tv, v[s], sizeof(double) * S.n, cudaMemcpyHostToDevice, h->stream);
      if (e != cudaSuccess) { cudaFree(tx); cudaFree(tv); return fail(set_err(h, PIC_ERR_CUDA, "upload v", e)); }
      dvp = tv;
    }
    rc = h->elem == 4 ? bin_species<float>(h, S, dxp, dvp) : bin_species<double>(h, S, dxp, dvp);
    cudaStreamSynchronize(h->stream);
    cudaFree(tx);
    cudaFree(tv);
    if (rc != PIC_OK) return fail(rc);
  }
  int32_t flag = 0;
  INIT_CUDA(cudaMemcpyAsync(&flag, h->d_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, h->stream));
  INIT_CUDA(cudaStreamSynchronize(h->stream));
  if (flag) return fail(set_err(h, PIC_ERR_PARTICLE, "particle with x outside [0,L) or non-finite x/v"));
  rc = mover_configure(h);
  if (rc != PIC_OK) return fail(rc);
  INIT_CUDA(cudaMalloc(&h->d_partial, sizeof(double) * (size_t)std::max(h->total_rows, 1) * ng));
#undef INIT_CUDA
  *out = h;
  return PIC_OK;
}

// a0-a8 for every species with the fields already on the device: launches only
static int move_device(pic_handle* h, const double* dEn, const double* dEp, double dt, double tol,
                       bool timed = true) {
  int rc;
  const int ns = (int)h->sp.size();
  PIC_CUDA(h, cudaMemsetAsync(h->d_queue, 0, sizeof(unsigned long long) * (ns + ST_COUNT), h->stream));
  if (timed) PIC_CUDA(h, cudaEventRecord(h->ev0, h->stream));
  int row = 0;
  for (int s = 0; s < ns; ++s) {
    if ((rc = launch_mover(h, s, dEn, dEp, dt, tol, row)) != PIC_OK) return rc;
    row += h->sp[s].last_blocks;
  }
  if (timed) PIC_CUDA(h, cudaEventRecord(h->ev1, h->stream));
  const int32_t ng = h->grid.n_cells;
  reduce_rows_kernel<<<(ng + kRedCols - 1) / kRedCols, dim3(kRedCols, kRedRows), 0, h->stream>>>(
      row, ng, h->d_partial, h->d_jbar);
  h->launches++;
  PIC_CUDA(h, cudaGetLastError());
  h->have_np1 = !(h->params.flags & PIC_FLAG_NO_STORE);
  return PIC_OK;
}

int pic_move_accumulate(pic_handle* h, const double* E_n, const double* E_np1, double dt,
                        double tol, double* jbar_out) {
  if (!h) return PIC_ERR_ARG;
  if (!E_n || !E_np1 || !(dt > 0.0) || !(tol >= 0.0)) return set_err(h, PIC_ERR_ARG, "pic_move_accumulate: bad argument");
  const double *dEn = nullptr, *dEp = nullptr;
  int rc;
  if ((rc = to_device(h, E_n, h->dE_n, &dEn)) != PIC_OK) return rc;
  if ((rc = to_device(h, E_np1, h->dE_np1, &dEp)) != PIC_OK) return rc;
  if ((rc = move_device(h, dEn, dEp, dt, tol)) != PIC_OK) return rc;
  const bool host_out = jbar_out && !is_device_ptr(jbar_out);
  unsigned long long capped = 0;
  if (host_out)   // rides on the synchronisation the host copy of jbar needs anyway
    PIC_CUDA(h, cudaMemcpyAsync(&capped, h->d_stats + ST_SUBSTEP_CAP, sizeof capped,
                                cudaMemcpyDeviceToHost, h->stream));
  if ((rc = from_device(h, h->d_jbar, jbar_out)) != PIC_OK) return rc;
  if (capped) return set_err(h, PIC_ERR_SUBSTEP_CAP, "particles cut off at max_substeps");
  return PIC_OK;
}

int pic_set_step(pic_handle* h, const double* E_n, double dt, double tol) {
  if (!h) return PIC_ERR_ARG;
  if (!E_n || !(dt > 0.0) || !(tol >= 0.0)) return set_err(h, PIC_ERR_ARG, "pic_set_step: bad argument");
  PIC_CUDA(h, cudaMemcpyAsync(h->dE_step, E_n, sizeof(double) * h->grid.n_cells,
                              is_device_ptr(E_n) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                              h->stream));
  h->step_dt = dt;
  h->step_tol = tol;
  h->have_step = true;
  return PIC_OK;
}

}  // extern "C"

// h_pin is the source of truly asynchronous H2D copies.  A call that returned without
// synchronising (host E in, DEVICE residual out) may still have its copy queued -- e.g. behind
// pic_commit's re-binning kernels -- when the next call wants to overwrite the buffer: that call
// would then evaluate the residual at the NEXT call's field.  Wait for the pending copy first.
static int pin_wait(pic_handle* h) {
  if (h->pin_busy) {
    PIC_CUDA(h, cudaEventSynchronize(h->ev_pin));
    h->pin_busy = false;
  }
  return PIC_OK;
}

// One residual evaluation from host E^{n+1} to host R as a CUDA graph, captured once per
// (flags, dt, tol, handle epoch) and replayed: at 1-4 M particles a pass is 0.1-0.2 ms of kernels, and the five
// launches, two copies and two event records around them were a quarter of its wall time.
// Returns PIC_ERR_UNSUPPORTED if the stream cannot be captured (the caller falls back).
static int residual_graph(pic_handle* h, const double* E_np1, double* resid_out) {
  const int32_t ng = h->grid.n_cells;
  cudaStream_t st = h->stream;
  if (!st) {   // the legacy default stream cannot be captured: a blocking stream of our own
    if (!h->own_stream && cudaStreamCreate(&h->own_stream) != cudaSuccess) {
      cudaGetLastError();
      return PIC_ERR_UNSUPPORTED;
    }
    st = h->own_stream;
  }
  double* out = h->h_pin + (ng + 1);
  pic_handle::ResidualGraph* g = nullptr;
  for (auto& e : h->graphs)
    if (e.flags == h->params.flags && e.dt == h->step_dt && e.tol == h->step_tol &&
        e.epoch == h->epoch)
      g = &e;
  if (!g) {
    if (h->graphs.size() >= 8) {
      for (auto& e : h->graphs) cudaGraphExecDestroy(e.exec);
      h->graphs.clear();
    }
    cudaStream_t user = h->stream;
    const long long l0 = h->launches;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
      cudaGetLastError();
      return PIC_ERR_UNSUPPORTED;
    }
    h->stream = st;
    int rc = PIC_OK;
    cudaError_t ce = cudaMemcpyAsync(h->dE_np1, h->h_pin, sizeof(double) * ng, cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) rc = move_device(h, h->dE_step, h->dE_np1, h->step_dt, h->step_tol, false);
    if (ce == cudaSuccess && rc == PIC_OK) {
      residual_kernel<<<1, 256, 0, st>>>(ng, h->dE_step, h->dE_np1, h->step_dt, h->d_jbar, h->d_resid,
                                         h->d_stats + ST_SUBSTEP_CAP);
      h->launches++;
      ce = cudaMemcpyAsync(out, h->d_resid, sizeof(double) * (ng + 1), cudaMemcpyDeviceToHost, st);
    }
    h->stream = user;
    cudaGraph_t graph = nullptr;
    cudaError_t ee = cudaStreamEndCapture(st, &graph);
    cudaGraphExec_t exec = nullptr;
    if (ce == cudaSuccess && rc == PIC_OK && ee == cudaSuccess && graph)
      ee = cudaGraphInstantiate(&exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    const long long nl = h->launches - l0;
    h->launches = l0;
    if (ce != cudaSuccess || rc != PIC_OK || ee != cudaSuccess || !exec) {
      cudaGetLastError();
      return PIC_ERR_UNSUPPORTED;
    }
    h->graphs.push_back({h->params.flags, h->step_dt, h->step_tol, exec, nl, h->epoch});
    g = &h->graphs.back();
  }
  if (int rc = pin_wait(h)) return rc;
  std::memcpy(h->h_pin, E_np1, sizeof(double) * ng);
  PIC_CUDA(h, cudaGraphLaunch(g->exec, st));
  h->launches += g->n_launches;
  h->have_np1 = !(h->params.flags & PIC_FLAG_NO_STORE);
  PIC_CUDA(h, cudaStreamSynchronize(st));
  std::memcpy(resid_out, out, sizeof(double) * ng);
  if (out[ng] != 0.0) return set_err(h, PIC_ERR_SUBSTEP_CAP, "particles cut off at max_substeps");
  return PIC_OK;
}

// pic_residual with the kind of each pointer known (1 = device, 0 = host, -1 = ask the driver):
// the JFNK driver calls it 13-36 times per time step with host arrays, so the host side is kept
// to one staged copy in, the launches, and one staged copy out that also carries the count of
// orbits cut off at max_substeps (A-9).
int picb200::residual_impl(pic_handle* h, const double* E_np1, double* resid_out, int e_dev, int r_dev) {
  if (!h) return PIC_ERR_ARG;
  if (!h->have_step) return set_err(h, PIC_ERR_STATE, "pic_residual before pic_set_step");
  if (!E_np1 || !resid_out) return set_err(h, PIC_ERR_ARG, "pic_residual: NULL argument");
  const int32_t ng = h->grid.n_cells;
  if (e_dev < 0) e_dev = is_device_ptr(E_np1) ? 1 : 0;
  if (r_dev < 0) r_dev = is_device_ptr(resid_out) ? 1 : 0;
  const double* dEp = E_np1;
  int rc;
  if (!e_dev && !r_dev && !h->graphs_off) {
    // host in, host out (the JFNK driver): the whole evaluation is one CUDA graph per
    // (flags, dt, tol) -- copy in, memset, movers, row sum, residual, copy out
    rc = residual_graph(h, E_np1, resid_out);
    if (rc != PIC_ERR_UNSUPPORTED) return rc;
    h->graphs_off = true;     // capture not possible here: plain launches
  }
  if (!e_dev) {
    if ((rc = pin_wait(h)) != PIC_OK) return rc;
    std::memcpy(h->h_pin, E_np1, sizeof(double) * ng);
    PIC_CUDA(h, cudaMemcpyAsync(h->dE_np1, h->h_pin, sizeof(double) * ng, cudaMemcpyHostToDevice, h->stream));
    if (r_dev) {   // this call will not synchronise: remember that the copy may still be pending
      PIC_CUDA(h, cudaEventRecord(h->ev_pin, h->stream));
      h->pin_busy = true;
    }
    dEp = h->dE_np1;
  }
  if ((rc = move_device(h, h->dE_step, dEp, h->step_dt, h->step_tol)) != PIC_OK) return rc;
  residual_kernel<<<1, 256, 0, h->stream>>>(ng, h->dE_step, dEp, h->step_dt, h->d_jbar, h->d_resid,
                                            h->d_stats + ST_SUBSTEP_CAP);
  h->launches++;
  PIC_CUDA(h, cudaGetLastError());
  if (r_dev) {
    PIC_CUDA(h, cudaMemcpyAsync(resid_out, h->d_resid, sizeof(double) * ng, cudaMemcpyDeviceToDevice, h->stream));
    return PIC_OK;     // no synchronisation, so no cap report (pic_get_stats has the count)
  }
  double* out = h->h_pin + (ng + 1);
  PIC_CUDA(h, cudaMemcpyAsync(out, h->d_resid, sizeof(double) * (ng + 1), cudaMemcpyDeviceToHost, h->stream));
  PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  std::memcpy(resid_out, out, sizeof(double) * ng);
  if (out[ng] != 0.0) return set_err(h, PIC_ERR_SUBSTEP_CAP, "particles cut off at max_substeps");
  return PIC_OK;
}

extern "C" {

int pic_residual(pic_handle* h, const double* E_np1, double* resid_out) {
  return picb200::residual_impl(h, E_np1, resid_out, -1, -1);
}

int pic_copy_state(pic_handle* dst, pic_handle* src) {
  if (!dst || !src) return PIC_ERR_ARG;
  if (dst == src) return PIC_OK;
  if (dst->grid.n_cells != src->grid.n_cells || dst->grid.length != src->grid.length ||
      dst->sp.size() != src->sp.size())
    return set_err(dst, PIC_ERR_ARG, "pic_copy_state: grids or species differ");
  for (size_t s = 0; s < src->sp.size(); ++s) {
    if (dst->sp[s].n != src->sp[s].n) return set_err(dst, PIC_ERR_ARG, "pic_copy_state: particle counts differ");
    // dst takes over src's sort key: its binning scratch (d_hist, d_scan) must hold that many keys
    const SpeciesState& A = src->sp[s];
    if ((long long)dst->grid.n_cells * A.nx * A.nv > dst->n_keys)
      return set_err(dst, PIC_ERR_ARG, "pic_copy_state: dst was created without PIC_FLAG_VSORT (or "
                                       "with fewer sort keys) than src's binning needs");
  }
  // src's pending work must be complete before dst's stream reads its buffers
  PIC_CUDA(dst, cudaStreamSynchronize(src->stream));
  for (size_t s = 0; s < src->sp.size(); ++s) {
    const SpeciesState& A = src->sp[s];
    SpeciesState& Bs = dst->sp[s];
    if (A.n == 0) continue;
    const int a = src->cur, b = dst->cur;
    if (src->elem == 8 && dst->elem == 4) {
      convert_arr<double, float>(dst, A.n, A.xi[a], Bs.xi[b]);
      convert_arr<double, float>(dst, A.n, A.v[a], Bs.v[b]);
    } else if (src->elem == 4 && dst->elem == 8) {
      convert_arr<float, double>(dst, A.n, A.xi[a], Bs.xi[b]);
      convert_arr<float, double>(dst, A.n, A.v[a], Bs.v[b]);
    } else {
      PIC_CUDA(dst, cudaMemcpyAsync(Bs.xi[b], A.xi[a], src->elem * A.n, cudaMemcpyDeviceToDevice, dst->stream));
      PIC_CUDA(dst, cudaMemcpyAsync(Bs.v[b], A.v[a], src->elem * A.n, cudaMemcpyDeviceToDevice, dst->stream));
    }
    PIC_CUDA(dst, cudaMemcpyAsync(Bs.cell[b], A.cell[a], sizeof(int32_t) * A.n, cudaMemcpyDeviceToDevice, dst->stream));
    PIC_CUDA(dst, cudaMemcpyAsync(Bs.id[b], A.id[a], sizeof(uint32_t) * A.n, cudaMemcpyDeviceToDevice, dst->stream));
    Bs.nx = A.nx; Bs.nv = A.nv; Bs.vmean = A.vmean; Bs.vinv = A.vinv; Bs.strided = A.strided;
  }
  PIC_CUDA(dst, cudaGetLastError());
  dst->have_np1 = false;
  // the sort key (nx, nv, strided) feeds launch arguments that captured residual graphs hold by
  // value (refill threshold): graphs of the old key are stale from here on
  dst->epoch++;
  for (auto& e : dst->graphs) cudaGraphExecDestroy(e.exec);
  dst->graphs.clear();
  return PIC_OK;
}

int pic_debug_bounds(int64_t* violations, int self_test) {
  if (!violations) return PIC_ERR_ARG;
#if PIC_BOUNDS_CHECK
  if (self_test) {
    int* d = nullptr;
    if (cudaMalloc(&d, 3 * sizeof(int)) != cudaSuccess) { cudaGetLastError(); return PIC_ERR_CUDA; }
    bounds_self_test_kernel<<<1, 1>>>(d);
    cudaDeviceSynchronize();
    cudaFree(d);
  }
  unsigned long long v = 0;
  if (cudaDeviceSynchronize() != cudaSuccess ||
      cudaMemcpyFromSymbol(&v, g_bounds_violations, sizeof v) != cudaSuccess) {
    cudaGetLastError();
    return PIC_ERR_CUDA;
  }
  *violations = (int64_t)v;
#else
  (void)self_test;
  *violations = -1;   // not the check build
#endif
  return PIC_OK;
}

int pic_commit(pic_handle* h) {
  if (!h) return PIC_ERR_ARG;
  if (!h->have_np1) return set_err(h, PIC_ERR_STATE, "pic_commit without a stored state n+1");
  for (auto& S : h->sp) {
    if (S.n == 0) continue;
    int rc = h->elem == 4 ? rebin_species<float>(h, S) : rebin_species<double>(h, S);
    if (rc != PIC_OK) return rc;
  }
  h->have_np1 = false;
  return PIC_OK;
}

}  // extern "C"
