// sm_100a kernels of hpsi_apply.  FP64 tensor path = mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), the only FP64 MMA
// sm_100a has (tcgen05 has no f64 kind); operands staged HBM/L2 -> shared memory with cp.async (LDGSTS),
// accumulators in registers.  One CTA = 1 producer warp + 2x2 consumer warps on a <=64x64 tile (<=4x4 fragments each).
#pragma once
#include <cuda_runtime.h>

#include "plan.h"

namespace hpsi {

constexpr int NCONS = 4;                       // consumer (DMMA) warps per CTA, 2 x 2 over the tile
constexpr int NTHREADS = (NCONS + 1) * 32;     // + 1 producer (cp.async) warp
constexpr int NSTAGE = 4;
// one stage: X[4 k-slabs][64 rows][4] and Y[4][64][4] doubles = 2 * 8 KB
constexpr int STAGE_DOUBLES = 2 * 4 * TILE * 4;
// stages | full[NSTAGE], empty[NSTAGE] mbarriers | 64 row pointers (P1)
constexpr int SMEM_BYTES = NSTAGE * STAGE_DOUBLES * 8 + 2 * NSTAGE * 8 + TILE * 8;

struct DevSchedule {           // device pointers to the uploaded tables
  const PsiBlk* blocks;
  const Seg* segs;
  const Group* groups;
  const P1Unit* p1;
  const Run* runs;
  const P2Unit* p2;
  const DiagTask* diag;
  double* ws;
  const double* a;
  const double* b;
  int n_blocks, n_p1, n_p2;
  int max_block_elems;
  int debug;                   // HPSI_DEBUG env (timing experiments only): 1 = producer skips loads, 2 = consumers skip MMAs
};

void launch_prep(const DevSchedule& d, const double* psi, cudaStream_t st);
void launch_p1(const DevSchedule& d, bool aligned16, cudaStream_t st);
void launch_p2(const DevSchedule& d, bool aligned16, cudaStream_t st);
void launch_reduce(const DevSchedule& d, double* out, cudaStream_t st);
void launch_diag(const DevSchedule& d, double* diag, cudaStream_t st);
cudaError_t kernels_init();    // opt-in to >48 KB dynamic shared memory

}  // namespace hpsi
