// pic_internal.h — handle layout and host-side helpers of the C-ABI library (not exported).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/pic.h"

namespace picb200 {

// One species' device state.  Two SoA buffers (state n / n+1), binned by cell.
struct SpeciesState {
  long long n = 0;
  double q_over_m = 0, w_q = 0;
  void* xi[2] = {nullptr, nullptr};       // T[n] in-cell offset, cell units
  void* v[2] = {nullptr, nullptr};        // T[n]
  int32_t* cell[2] = {nullptr, nullptr};  // int32[n]
  uint32_t* id[2] = {nullptr, nullptr};   // original index of the particle in each slot
  uint32_t* nsub = nullptr;               // optional per-particle counts of the last move
  uint32_t* ncross = nullptr;
  int32_t nx = 1, nv = 1;                 // offset / velocity classes of the sort key (1 = cell only)
  double vmean = 0, vinv = 0;
  bool strided = false;                   // PIC_FLAG_STRIDED: (v class, offset class, cell) order
  int grid_blocks = 0;                    // mover launch shape for this species
  int grid_blocks2 = 0;                   // same for the two-per-lane fp32 kernel (0 = not usable)
  int last_blocks = 0;                    // blocks (= rows of `partial`) of the last launch
  int tile = 0;
  int tile2 = 0;
};

}  // namespace picb200

struct pic_handle {
  pic_grid grid{};
  pic_params params{};
  std::vector<picb200::SpeciesState> sp;
  cudaStream_t stream = nullptr;
  int cur = 0;                 // index of the buffer holding state n
  bool have_np1 = false;       // a move has produced state n+1 since the last commit
  bool have_step = false;      // pic_set_step was called
  double step_dt = 0, step_tol = 0;
  size_t elem = 4;             // sizeof(T)
  int sm_count = 0;
  int blocks_per_sm = 2;
  size_t smem_bytes = 0;
  size_t smem_bytes2 = 0;      // two-per-lane fp32 kernel (mover2.cuh)
  // device scratch
  double* dE_n = nullptr;      // [n_cells] staging for host E^n / stored E^n of pic_set_step
  double* dE_step = nullptr;   // [n_cells] E^n of pic_set_step
  double* dE_np1 = nullptr;
  double* d_jbar = nullptr;
  double* d_resid = nullptr;
  unsigned char* d_grid_scratch = nullptr;  // large grids: per-block grid copies in global memory
  size_t grid_stride = 0;
  int ggrid_max_blocks = 0;
  double* d_partial = nullptr; // [total_rows][n_cells]
  int total_rows = 0;
  unsigned long long* d_queue = nullptr;  // [n_species] + [ST_COUNT]: one allocation, one memset
  unsigned long long* d_stats = nullptr;  // = d_queue + n_species
  double* h_pin = nullptr;                // pinned host staging, 2 x (n_cells + 1)
  cudaEvent_t ev_pin = nullptr;           // recorded after an H2D copy out of h_pin that no
  bool pin_busy = false;                  // synchronisation follows: wait before h_pin is rewritten
  int32_t* d_hist = nullptr;              // [n_keys + 1] binning scratch
  long long n_keys = 0;
  int32_t* d_scan = nullptr;              // [n_keys / 4096 + 1] chunk sums of the scan
  int32_t* d_flag = nullptr;              // validation flag
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  // CUDA graphs of one residual evaluation with host vectors (pic_api.cu: residual_impl)
  struct ResidualGraph {
    uint32_t flags;
    double dt, tol;
    cudaGraphExec_t exec;
    long long n_launches;
    long long epoch;                   // handle epoch the kernel arguments were captured in
  };
  std::vector<ResidualGraph> graphs;
  cudaStream_t own_stream = nullptr;   // for graph launches when `stream` is the legacy default stream
  bool graphs_off = false;             // a capture failed once: plain launches from then on
  long long epoch = 0;                 // bumped by whatever changes launch arguments a graph bakes
                                       // in besides (flags, dt, tol): pic_copy_state (sort key)
  pic_stats stats{};
  long long launches = 0;
  const char* last_kernel = "";   // name of the mover kernel of the last launch
  std::string err;
};

namespace picb200 {

int set_err(pic_handle* h, int code, const char* what, cudaError_t ce = cudaSuccess);
bool is_device_ptr(const void* p);
// mover launch (pic_mover.cu)
int launch_mover(pic_handle* h, int s, const double* dE_n, const double* dE_np1, double dt,
                 double tol, int row0);
int mover_configure(pic_handle* h);
// pic_residual with known pointer kinds (1 device, 0 host, -1 unknown); pic_api.cu
int residual_impl(pic_handle* h, const double* E_np1, double* resid_out, int e_dev, int r_dev);

}  // namespace picb200

#define PIC_CUDA(h, call)                                                        \
  do {                                                                           \
    cudaError_t ce_ = (call);                                                    \
    if (ce_ != cudaSuccess) return picb200::set_err((h), PIC_ERR_CUDA, #call, ce_); \
  } while (0)
