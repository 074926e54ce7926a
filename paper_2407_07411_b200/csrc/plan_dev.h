// The opaque hpsi_plan: host schedule + its device copy + plan-owned device buffers.
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "kernels.cuh"
#include "plan.h"

struct hpsi_plan {
  hpsi::Schedule sc;
  bool host_only = false;
  bool device_ok = false;         // a CUDA device was initialised for this plan: device buffers may exist and must be freed
  bool bound = false;
  bool aligned16 = true;          // descriptors AND arena bases have 16-byte aligned rows: TMA staging is used
  int n_sm = 148;
  hpsi::DevSchedule dev{};
  void* d_tables = nullptr;       // one allocation holding every uploaded table
  double* d_ws = nullptr;
  void* d_maps = nullptr;         // CUtensorMap[sc.maps.size()], encoded by hpsi_bind
  // apply_host staging
  double* d_psi_stage = nullptr;
  double* d_out_stage = nullptr;
  // Davidson buffers (allocated on first use)
  double* d_dav = nullptr;
  size_t dav_doubles = 0;
  int dav_mmax = 0;
  double* h_dav = nullptr;        // pinned host scalars the Davidson loop reads back each iteration
  cudaStream_t dav_side = nullptr;   // side stream + events: the read-back of an iteration's residual overlaps its
  cudaEvent_t dav_ev[2] = {nullptr, nullptr};   // orthogonalisation kernels (davidson.cu)
  // hpsi_set_exchange: called by the eigensolvers after every mat-vec / diagonal they compute (term-sharded plans)
  hpsi_exchange_fn exchange_fn = nullptr;
  void* exchange_user = nullptr;
  // hpsi_truncate (svd.cu)
  int n_left = 0, n_right = 0;    // sectors of the sector table (length of chi_host for either side)
  void* d_svd = nullptr;          // working matrices, singular values, tables (allocated on first use)
  size_t svd_bytes = 0;
  int svd_sweeps = 0, svd_launches = 0;   // of the last hpsi_truncate call (diagnostics)
};

namespace hpsi {
void set_error(const std::string& s);
int cuda_fail(cudaError_t e, const char* what);   // records the message, returns HPSI_ECUDA
int apply_impl(hpsi_plan_t* p, const double* psi_dev, double* out_dev, bool accumulate, void* cuda_stream,
               const double* nrm2_dev = nullptr, double* normalized_dev = nullptr,   // out = H (psi / sqrt(nrm2[v])), see prep_kernel
               int n_vectors = 1, int64_t ld_psi = 0, int64_t ld_out = 0);             // batched plans: vectors ld_* doubles apart
// api.cu: shared with rotate.cu, whose object wraps an hpsi_plan
int upload_schedule(hpsi_plan_t* p);   // device copies of the schedule tables, workspace, tensor-map buffer
int encode_maps(hpsi_plan_t* p);       // CUtensorMap of every MapSpec against dev.a / dev.b / d_ws
void free_plan(hpsi_plan_t* p);
}  // namespace hpsi

// CUDA events that are destroyed on every return path
template <int N>
struct EventSet {
  cudaEvent_t ev[N] = {};
  cudaError_t create() {
    for (auto& e : ev) { cudaError_t rc = cudaEventCreate(&e); if (rc != cudaSuccess) return rc; }
    return cudaSuccess;
  }
  ~EventSet() { for (auto& e : ev) if (e) cudaEventDestroy(e); }
  cudaEvent_t& operator[](int i) { return ev[i]; }
};

#define HPSI_CUDA(call)                                             \
  do {                                                              \
    cudaError_t e_ = (call);                                        \
    if (e_ != cudaSuccess) return hpsi::cuda_fail(e_, #call);       \
  } while (0)
