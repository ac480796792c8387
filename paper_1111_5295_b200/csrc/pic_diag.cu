// pic_diag.cu — getters and diagnostics of the C-ABI (include/pic.h): particle read-back in the
// original order, counts, totals, kinetic energy, rho.  Not on the hot path.
#include <algorithm>
#include <cstdio>
#include <cstring>

#include "mover.cuh"
#include "pic_internal.h"
#include "pic_kernels.cuh"

using namespace picb200;

namespace {

int grid_for(long long n) {
  long long g = (n + 255) / 256;
  return (int)std::max<long long>(1, std::min<long long>(g, 148 * 16));
}

// RAII device temporary used when the caller's output pointer is a host pointer.
template <typename U>
struct DevOut {
  U* user = nullptr;
  U* dev = nullptr;
  bool temp = false;
  size_t n = 0;
  cudaError_t prepare(U* p, size_t count) {
    user = p; n = count;
    if (!p) return cudaSuccess;
    if (is_device_ptr(p)) { dev = p; return cudaSuccess; }
    temp = true;
    return cudaMalloc(&dev, sizeof(U) * std::max<size_t>(count, 1));
  }
  cudaError_t finish(cudaStream_t st) {
    if (!temp || !user) return cudaSuccess;
    return cudaMemcpyAsync(user, dev, sizeof(U) * n, cudaMemcpyDeviceToHost, st);
  }
  ~DevOut() { if (temp) cudaFree(dev); }
};

}  // namespace

extern "C" {

int pic_get_particles(pic_handle* h, int species, int which, double* x, double* v,
                      int32_t* cell, double* xi) {
  if (!h) return PIC_ERR_ARG;
  if (species < 0 || species >= (int)h->sp.size() || (which != PIC_STATE_N && which != PIC_STATE_NP1))
    return set_err(h, PIC_ERR_ARG, "pic_get_particles: bad species/which");
  if (which == PIC_STATE_NP1 && !h->have_np1)
    return set_err(h, PIC_ERR_STATE, "pic_get_particles: no state n+1 (move not run or NO_STORE)");
  const SpeciesState& S = h->sp[species];
  if (S.n == 0) return PIC_OK;
  const int b = which == PIC_STATE_N ? h->cur : 1 - h->cur;
  DevOut<double> ox, ov, oxi;
  DevOut<int32_t> oc;
  PIC_CUDA(h, ox.prepare(x, S.n));
  PIC_CUDA(h, ov.prepare(v, S.n));
  PIC_CUDA(h, oxi.prepare(xi, S.n));
  PIC_CUDA(h, oc.prepare(cell, S.n));
  const double dx = h->grid.length / h->grid.n_cells;
  if (h->elem == 4)
    unpermute_kernel<float><<<grid_for(S.n), 256, 0, h->stream>>>(
        S.n, S.id[h->cur], (const float*)S.xi[b], (const float*)S.v[b], S.cell[b], dx, ox.dev,
        ov.dev, oc.dev, oxi.dev);
  else
    unpermute_kernel<double><<<grid_for(S.n), 256, 0, h->stream>>>(
        S.n, S.id[h->cur], (const double*)S.xi[b], (const double*)S.v[b], S.cell[b], dx, ox.dev,
        ov.dev, oc.dev, oxi.dev);
  h->launches++;
  PIC_CUDA(h, cudaGetLastError());
  PIC_CUDA(h, ox.finish(h->stream));
  PIC_CUDA(h, ov.finish(h->stream));
  PIC_CUDA(h, oxi.finish(h->stream));
  PIC_CUDA(h, oc.finish(h->stream));
  PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  return PIC_OK;
}

int pic_get_counts(pic_handle* h, int species, uint32_t* n_sub, uint32_t* n_cross) {
  if (!h) return PIC_ERR_ARG;
  if (species < 0 || species >= (int)h->sp.size())
    return set_err(h, PIC_ERR_ARG, "pic_get_counts: bad species");
  const SpeciesState& S = h->sp[species];
  if (!S.nsub || !(h->params.flags & PIC_FLAG_COUNTS))
    return set_err(h, PIC_ERR_STATE, "pic_get_counts: PIC_FLAG_COUNTS was not set at pic_init");
  if (S.n == 0) return PIC_OK;
  DevOut<uint32_t> oa, ob;
  PIC_CUDA(h, oa.prepare(n_sub, S.n));
  PIC_CUDA(h, ob.prepare(n_cross, S.n));
  unpermute_counts_kernel<<<grid_for(S.n), 256, 0, h->stream>>>(S.n, S.id[h->cur], S.nsub,
                                                                S.ncross, oa.dev, ob.dev);
  h->launches++;
  PIC_CUDA(h, cudaGetLastError());
  PIC_CUDA(h, oa.finish(h->stream));
  PIC_CUDA(h, ob.finish(h->stream));
  PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  return PIC_OK;
}

int pic_count_histogram(pic_handle* h, int species, uint32_t bin_width, int32_t n_bins,
                        unsigned long long* hist_sub, unsigned long long* hist_cross) {
  if (!h) return PIC_ERR_ARG;
  if (species < 0 || species >= (int)h->sp.size() || bin_width < 1 || n_bins < 1 ||
      n_bins > kHistMaxBins)
    return set_err(h, PIC_ERR_ARG, "pic_count_histogram: bad argument");
  const SpeciesState& S = h->sp[species];
  if (!S.nsub || !(h->params.flags & PIC_FLAG_COUNTS))
    return set_err(h, PIC_ERR_STATE, "pic_count_histogram: PIC_FLAG_COUNTS was not set at pic_init");
  unsigned long long* d = nullptr;
  const size_t bytes = sizeof(unsigned long long) * (size_t)n_bins;
  PIC_CUDA(h, cudaMalloc(&d, 2 * bytes));
  cudaError_t e = cudaMemsetAsync(d, 0, 2 * bytes, h->stream);
  if (e == cudaSuccess && S.n > 0) {
    const int blocks = (int)std::min<long long>((S.n + 255) / 256, 4LL * h->sm_count);
    const size_t sm = sizeof(uint32_t) * (size_t)n_bins;
    count_hist_kernel<<<blocks, 256, sm, h->stream>>>(S.n, S.nsub, bin_width, n_bins, d);
    count_hist_kernel<<<blocks, 256, sm, h->stream>>>(S.n, S.ncross, bin_width, n_bins, d + n_bins);
    h->launches += 2;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess && hist_sub)
    e = cudaMemcpyAsync(hist_sub, d, bytes, cudaMemcpyDefault, h->stream);
  if (e == cudaSuccess && hist_cross)
    e = cudaMemcpyAsync(hist_cross, d + n_bins, bytes, cudaMemcpyDefault, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  cudaFree(d);
  if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "pic_count_histogram", e);
  return PIC_OK;
}

int pic_get_stats(pic_handle* h, pic_stats* out) {
  if (!h || !out) return PIC_ERR_ARG;
  unsigned long long st[ST_COUNT];
  PIC_CUDA(h, cudaMemcpyAsync(st, h->d_stats, sizeof st, cudaMemcpyDeviceToHost, h->stream));
  PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  pic_stats& s = h->stats;
  s.n_sub = (int64_t)st[ST_SUB];
  s.n_cross = (int64_t)st[ST_CROSS];
  s.n_picard_it = (int64_t)st[ST_PICARD_IT];
  s.n_picard_cap = (int64_t)st[ST_PICARD_CAP];
  s.n_kappa_cap = (int64_t)st[ST_KAPPA_CAP];
  s.n_substep_cap = (int64_t)st[ST_SUBSTEP_CAP];
  s.n_neg_disc = (int64_t)st[ST_NEG_DISC];
  s.n_clamped_tau = (int64_t)st[ST_CLAMPED];
  s.n_launches = h->launches;
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, h->ev0, h->ev1) != cudaSuccess) { cudaGetLastError(); ms = 0.f; }
  s.last_move_ms = ms;
  *out = s;
  return PIC_OK;
}

int pic_set_flags(pic_handle* h, uint32_t flags) {
  if (!h) return PIC_ERR_ARG;
  if ((flags & PIC_FLAG_COUNTS) && !h->sp.empty() && !h->sp[0].nsub)
    return set_err(h, PIC_ERR_STATE, "PIC_FLAG_COUNTS must be set at pic_init (buffers)");
  // the global-memory-grid kernels (grids beyond a block's shared memory) exist with the
  // end-point deposit and plain fp32 time accounting only: say so instead of ignoring the request
  if (h->d_grid_scratch) {
    if (flags & PIC_FLAG_DEPOSIT_PER_VISIT)
      return set_err(h, PIC_ERR_UNSUPPORTED, "pic_set_flags: per-visit deposit needs the grid in shared memory (n_cells too large)");
    if ((flags & PIC_FLAG_EXACT_TIME) && h->elem == 4)
      return set_err(h, PIC_ERR_UNSUPPORTED, "pic_set_flags: exact time accounting is not built for grids beyond shared memory (n_cells too large)");
  }
  h->params.flags = flags;
  return PIC_OK;
}

int pic_kinetic_energy(pic_handle* h, int which, double* ke_out) {
  if (!h || !ke_out) return PIC_ERR_ARG;
  if (which == PIC_STATE_NP1 && !h->have_np1)
    return set_err(h, PIC_ERR_STATE, "pic_kinetic_energy: no state n+1");
  const int ns = (int)h->sp.size();
  double* d = nullptr;
  PIC_CUDA(h, cudaMalloc(&d, sizeof(double) * ns));
  cudaMemsetAsync(d, 0, sizeof(double) * ns, h->stream);
  const int b = which == PIC_STATE_N ? h->cur : 1 - h->cur;
  for (int s = 0; s < ns; ++s) {
    const SpeciesState& S = h->sp[s];
    if (S.n == 0) continue;
    if (h->elem == 4)
      sumsq_kernel<float><<<grid_for(S.n), 256, 0, h->stream>>>(S.n, (const float*)S.v[b], d + s);
    else
      sumsq_kernel<double><<<grid_for(S.n), 256, 0, h->stream>>>(S.n, (const double*)S.v[b], d + s);
    h->launches++;
  }
  cudaError_t e = cudaMemcpyAsync(ke_out, d, sizeof(double) * ns, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  cudaFree(d);
  if (e != cudaSuccess) return set_err(h, PIC_ERR_CUDA, "pic_kinetic_energy", e);
  for (int s = 0; s < ns; ++s) ke_out[s] *= 0.5 * h->sp[s].w_q / h->sp[s].q_over_m;  // w_m/2
  return PIC_OK;
}

// persistent grid: a few blocks per SM, fewer for small species (>= one full pass per block)
static int rho_grid(const pic_handle* h, long long n) {
  const long long want = (n + 512LL * kRhoChunk - 1) / (512LL * kRhoChunk);
  return (int)std::max<long long>(1, std::min<long long>(want, 4LL * h->sm_count));
}

int pic_rho(pic_handle* h, int which, double* rho_out) {
  if (!h || !rho_out) return PIC_ERR_ARG;
  if (which == PIC_STATE_NP1 && !h->have_np1)
    return set_err(h, PIC_ERR_STATE, "pic_rho: no state n+1");
  const int32_t ng = h->grid.n_cells;
  const double dx = h->grid.length / ng;
  const int b = which == PIC_STATE_N ? h->cur : 1 - h->cur;
  PIC_CUDA(h, cudaMemsetAsync(h->d_resid, 0, sizeof(double) * ng, h->stream));
  size_t rho_smem = sizeof(double) * (size_t)ng;
  const bool rho_global = rho_smem > 200 * 1024;   // large grid: no shared-memory copy of rho
  if (rho_global) rho_smem = 0;
  if (rho_smem > 48 * 1024) {
    PIC_CUDA(h, cudaFuncSetAttribute(rho_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rho_smem));
    PIC_CUDA(h, cudaFuncSetAttribute(rho_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rho_smem));
  }
  for (auto& S : h->sp) {
    if (S.n == 0) continue;
    if (rho_global) {
      if (h->elem == 4)
        rho_kernel<float, false><<<rho_grid(h, S.n), 512, 0, h->stream>>>(
            S.n, (const float*)S.xi[b], S.cell[b], ng, S.w_q / dx, h->d_resid);
      else
        rho_kernel<double, false><<<rho_grid(h, S.n), 512, 0, h->stream>>>(
            S.n, (const double*)S.xi[b], S.cell[b], ng, S.w_q / dx, h->d_resid);
    } else if (h->elem == 4)
      rho_kernel<float><<<rho_grid(h, S.n), 512, rho_smem, h->stream>>>(S.n, (const float*)S.xi[b], S.cell[b],
                                                              ng, S.w_q / dx, h->d_resid);
    else
      rho_kernel<double><<<rho_grid(h, S.n), 512, rho_smem, h->stream>>>(S.n, (const double*)S.xi[b],
                                                               S.cell[b], ng, S.w_q / dx, h->d_resid);
    h->launches++;
  }
  PIC_CUDA(h, cudaGetLastError());
  const bool dev = is_device_ptr(rho_out);
  PIC_CUDA(h, cudaMemcpyAsync(rho_out, h->d_resid, sizeof(double) * ng,
                              dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  if (!dev) PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  return PIC_OK;
}

int pic_destroy(pic_handle* h) {
  if (!h) return PIC_OK;
  cudaStreamSynchronize(h->stream);
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
  delete h;
  return PIC_OK;
}

const char* pic_last_error(const pic_handle* h) { return h ? h->err.c_str() : "invalid handle"; }
const char* pic_last_kernel(const pic_handle* h) { return h ? h->last_kernel : ""; }

int pic_version(char* buf, int buflen) {
  if (!buf || buflen < 1) return PIC_ERR_ARG;
  int dev = -1;
  cudaDeviceProp prop;
  const char* name = "no CUDA device";
  int sms = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && cudaGetDeviceProperties(&prop, dev) == cudaSuccess) {
    name = prop.name;
    sms = prop.multiProcessorCount;
  } else {
    cudaGetLastError();
  }
  snprintf(buf, (size_t)buflen, "pic_b200 0.1 (sm_100a; block %d) on %s, %d SMs", kBlock, name, sms);
  return PIC_OK;
}

}  // extern "C"
