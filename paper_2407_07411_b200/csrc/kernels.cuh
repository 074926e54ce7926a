// sm_100a kernels of hpsi_apply.  FP64 tensor path = mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), the only FP64 MMA
// sm_100a has (tcgen05 has no f64 kind), accumulators in registers.  Operands are staged into shared memory by the
// TMA unit (cp.async.bulk.tensor.2d with one tensor map per operand matrix, 128-byte swizzle, zero fill out of
// bounds) when every block has 16-byte aligned rows; otherwise by 8-byte cp.async (LDGSTS) into the same layout.
// One CTA = 1 producer warp + 4 consumer warps on a <=64x64 tile (<=16 fragments each).
#pragma once
#include <cuda_runtime.h>

#include "plan.h"

namespace hpsi {

// Programmatic dependent launch (PDL).  A kernel launched with launch_dependent() may be set up on the GPU while the kernel
// before it in the stream is still running; it must call pdl_wait() before it touches global memory - the call returns
// when that kernel has completed and its writes are visible (a no-op after a plain launch).  No kernel here triggers its
// dependents early (an early trigger lets the next grid's CTAs occupy the SMs while this one still needs them: measured
// 2.3x slower on a 256-block chain), so the gain is the launch latency of every kernel boundary: 4.1 -> 2.3 us per
// boundary on B200, four boundaries per apply and nine per Davidson iteration - visible at D <= 1024 only.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <class... KArgs, class... Args>
inline cudaError_t launch_dependent(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                    Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

constexpr int NCONS = NCONS_WARPS;                     // consumer (DMMA) warps per CTA, as a 2x2, 1x4 or 4x1 grid over the tile
constexpr int NTHREADS = (NCONS + 1) * 32;     // + 1 producer warp
constexpr int CTAS_PER_SM = 3;
constexpr int NSTAGE = 4;
constexpr int OP_BYTES = TILE * KT * 8;        // one TMA box: 64 rows x 128 bytes, 128-byte swizzled
constexpr int X_BOXES = TILE_M / TILE;         // the X tile of a stage is X_BOXES boxes one under the other
constexpr int STAGE_BYTES = (X_BOXES + 1) * OP_BYTES;   // X tile | Y tile
// 1024 bytes of slack to align the stages (the swizzle pattern is a function of address bits 4-9) | stages | barriers
constexpr int SMEM_BYTES = 1024 + NSTAGE * STAGE_BYTES + 2 * NSTAGE * 8;
constexpr int TMAP_BYTES = 128;                // sizeof(CUtensorMap)

struct DevSchedule {           // device pointers to the uploaded tables
  const PsiBlk* blocks;
  const Seg* segs;
  const Group* groups;
  const P1Unit* p1;
  const Run* runs;
  const P2Unit* p2;
  const P2Unit* pf;            // fused units (kernels_fused.cu)
  const DiagTask* diag;
  const ElemCta* elem;         // granules of the element-wise kernels
  int n_elem;
  const unsigned char* maps;   // CUtensorMap[sc.maps.size()], 128 bytes each (TMA staging only)
  double* ws;
  const double* a;
  const double* b;
  int n_blocks, n_p1, n_p2, n_pf;
  int max_block_elems;
  int paired;                  // the plan has blocks stored transposed: kernels_paired.cu runs the GEMMs
  int nvec;                    // vectors the plan was laid out for (batched plans: hpsi_plan_options_t.n_vectors)
  int nvec_active;             // vectors of THIS apply (<= nvec): units of the others return at once
  int64_t ld_psi, ld_out;      // doubles between consecutive vectors of psi / out (hpsi_apply_multi)
  double* rot_dst;             // operator-update launches (rotate.cu) only: base the transposed tile stores go to
};

void launch_prep(const DevSchedule& d, const double* psi, const double* nrm2, double* normalized, cudaStream_t st);   // nrm2 != null: psi / sqrt(*nrm2), also written to `normalized`
void launch_p1(const DevSchedule& d, bool tma, cudaStream_t st);
void launch_p1_rot(const DevSchedule& d, bool tma, cudaStream_t st);   // same kernel, tile stored transposed at Seg.p2_off / p2_ld
void launch_p2(const DevSchedule& d, bool tma, cudaStream_t st);
void launch_pf(const DevSchedule& d, bool tma, cudaStream_t st);            // kernels_fused.cu
cudaError_t kernels_fused_init();
void launch_reduce(const DevSchedule& d, double* out, bool accumulate, cudaStream_t st);
void launch_diag(const DevSchedule& d, double* diag, cudaStream_t st);
void launch_sum_shards(const double* parts, int n_parts, int64_t n, double* out, cudaStream_t st);
void launch_p1_paired(const DevSchedule& d, bool tma, cudaStream_t st);   // kernels_paired.cu
void launch_p2_paired(const DevSchedule& d, bool tma, cudaStream_t st);
cudaError_t kernels_paired_init();
cudaError_t kernels_init();    // opt-in to >48 KB dynamic shared memory

}  // namespace hpsi
