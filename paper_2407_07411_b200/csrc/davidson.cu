// hpsi_davidson: Davidson-Liu, lowest eigenpair, single root (PAPER.md:62 names "Lanczos or Davidson"; the algorithm
// is DESIGN.md reading A21).  Every O(psi_length) operation and the small subspace eigenproblem (cyclic Jacobi in one
// warp) run on the device; the host reads back two scalars per iteration (residual norm^2, |s|^2) to steer the loop.
// All reductions are two-stage with a fixed order, so a run is bitwise reproducible.
#include <algorithm>
#include <cmath>

#include "plan_dev.h"

namespace {

constexpr int NB = 256;       // partial blocks per dot product
constexpr int MMAX = 32;

// out[v*stride] (and mirror[v*mstride] if given) = X_v . y for the nvec vectors X_v = X + v*ldx.
// Two stages in one launch: block (b, v) reduces its slice into partial[v][b]; the block that finishes last for vector v
// (ticket from an atomic counter - control only) adds the NB partials in a fixed order, so the result does not depend
// on which block that is and a run is bitwise reproducible.  The counter is left at zero for the next call.
__global__ void dot_kernel(const double* __restrict__ X, int64_t ldx, const double* __restrict__ y, int64_t n,
                           double* __restrict__ partial, unsigned int* __restrict__ counters, double* out, int stride,
                           double* mirror, int mstride) {
  __shared__ double red[256];
  __shared__ bool last;
  const int v = blockIdx.y;
  const double* x = X + (int64_t)v * ldx;
  const int64_t per = (n + NB - 1) / NB;
  const int64_t lo = (int64_t)blockIdx.x * per, hi = (lo + per < n) ? lo + per : n;
  double s = 0.0;
  for (int64_t e = lo + threadIdx.x; e < hi; e += 256) s += x[e] * y[e];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    partial[v * NB + blockIdx.x] = red[0];
    __threadfence();
    last = atomicAdd(counters + v, 1u) == NB - 1;
  }
  __syncthreads();
  if (!last || threadIdx.x >= 32) return;
  __threadfence();
  double t = 0.0;                                        // lane l: partials 8l .. 8l+7 in order, then a fixed shuffle tree
  const volatile double* pv = partial + v * NB + threadIdx.x * (NB / 32);
  for (int i = 0; i < NB / 32; ++i) t += pv[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  if (threadIdx.x == 0) {
    out[(int64_t)v * stride] = t;
    if (mirror) mirror[(int64_t)v * mstride] = t;
    counters[v] = 0;
  }
}

// dst = src / sqrt(*nrm2)   (dst2 = src2 / sqrt(*nrm2) if given)
__global__ void scale_kernel(double* dst, const double* src, double* dst2, const double* src2, const double* nrm2,
                             int64_t n) {
  const double inv = 1.0 / sqrt(*nrm2);
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    dst[e] = src[e] * inv;
    if (dst2) dst2[e] = src2[e] * inv;
  }
}

// Smallest eigenpair of the symmetric j x j matrix G (leading dimension MMAX) by parallel two-sided Jacobi: the j/2
// disjoint rotations of a round-robin round are applied together, warp k = pair k, lane t = row t (blockDim.x =
// 32 * ceil(j/2)); first all column updates A J, then all row updates J^T (A J).  (A one-warp cyclic version took 86 us per
// call at j ~ 10 - a quarter of a Davidson iteration's fixed cost.)  Writes theta[0] and y[0..j); G is left untouched.
__global__ void small_eig_kernel(const double* __restrict__ G, int j, double* theta, double* y) {
  __shared__ double A[MMAX][MMAX + 1], Q[MMAX][MMAX + 1];
  __shared__ double norms[2];
  const int t = threadIdx.x & 31, k = threadIdx.x >> 5;
  const int m = (j + 1) & ~1;                            // players of the round-robin (a dummy one if j is odd)
  const int np = m > 1 ? m / 2 : 1;                      // = warps in the block
  for (int c = k; c < j; c += np)
    if (t < j) { A[t][c] = 0.5 * (G[t * MMAX + c] + G[c * MMAX + t]); Q[t][c] = (t == c) ? 1.0 : 0.0; }
  __syncthreads();
  for (int sweep = 0; sweep < 30 && j > 1; ++sweep) {
    if (k == 0) {                                        // squared norms of the off-diagonal part and of the diagonal
      double off = 0.0, dg = 0.0;
      if (t < j) {
        dg = A[t][t] * A[t][t];
        for (int q = t + 1; q < j; ++q) off += A[t][q] * A[t][q];
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dg += __shfl_xor_sync(0xffffffffu, dg, o); }
      if (t == 0) { norms[0] = off; norms[1] = dg; }
    }
    __syncthreads();
    const double off = norms[0], dg = norms[1];
    if (off <= 1e-34 * (dg + 2.0 * off) || off < 1e-300) break;   // off-diagonal norm below 1e-17 of the matrix norm
    for (int r = 0; r < m - 1; ++r) {
      int p, q;
      if (k == 0) { p = m - 1; q = r; }
      else { p = (r + k) % (m - 1); q = (r - k + m - 1) % (m - 1); }
      if (p > q) { const int tmp = p; p = q; q = tmp; }
      double c = 1.0, sn = 0.0;
      if (q < j) {                                       // not the dummy player
        const double apq = A[p][q];
        if (fabs(apq) >= 1e-300) {
          const double app = A[p][p], aqq = A[q][q];
          const double tau = (aqq - app) / (2.0 * apq);
          const double tt = (tau >= 0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
          c = 1.0 / sqrt(1.0 + tt * tt);
          sn = tt * c;
        }
      }
      __syncwarp();
      const bool act = sn != 0.0 && t < j;
      if (act) {                                         // columns p, q (this warp's alone)
        const double akp = A[t][p], akq = A[t][q];
        A[t][p] = c * akp - sn * akq;
        A[t][q] = sn * akp + c * akq;
        const double qkp = Q[t][p], qkq = Q[t][q];
        Q[t][p] = c * qkp - sn * qkq;
        Q[t][q] = sn * qkp + c * qkq;
      }
      __syncthreads();
      if (act) {                                         // rows p, q
        const double apk = A[p][t], aqk = A[q][t];
        A[p][t] = c * apk - sn * aqk;
        A[q][t] = sn * apk + c * aqk;
      }
      __syncthreads();
    }
  }
  __syncthreads();
  if (k == 0) {
    int best = 0;
    for (int i = 1; i < j; ++i)
      if (A[i][i] < A[best][best]) best = i;
    if (t == 0) theta[0] = A[best][best];
    if (t < j) y[t] = Q[t][best];
  }
}

// x = sum_i y_i V_i ; wy = sum_i y_i W_i ; r = wy - theta x
__global__ void ritz_kernel(const double* __restrict__ V, const double* __restrict__ W, int64_t n, int j,
                            const double* __restrict__ y, const double* __restrict__ theta, double* x, double* wy,
                            double* r) {
  const double th = *theta;
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double sx = 0.0, sw = 0.0;
    for (int i = 0; i < j; ++i) { const double yi = y[i]; sx += yi * V[i * n + e]; sw += yi * W[i * n + e]; }
    x[e] = sx; wy[e] = sw; r[e] = sw - th * sx;
  }
}

// s = r / (diag - theta) with |den| clamped to >= 1e-8 keeping its sign; or s = r
__global__ void precond_kernel(const double* __restrict__ r, const double* __restrict__ diag,
                               const double* __restrict__ theta, int precondition, double* s, int64_t n) {
  const double th = *theta;
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double v = r[e];
    if (precondition) {
      double den = diag[e] - th;
      if (fabs(den) < 1e-8) den = (den < 0) ? -1e-8 : 1e-8;
      v /= den;
    }
    s[e] = v;
  }
}

// s -= sum_i c_i V_i
__global__ void project_kernel(double* s, const double* __restrict__ V, int64_t n, int j, const double* __restrict__ c) {
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double acc = s[e];
    for (int i = 0; i < j; ++i) acc -= c[i] * V[i * n + e];
    s[e] = acc;
  }
}

__global__ void set_scalar_kernel(double* dst, const double* src) { *dst = *src; }

}  // namespace

extern "C" int hpsi_davidson(hpsi_plan_t* p, double* psi, double* eig_host, const hpsi_davidson_params_t* params,
                             hpsi_davidson_info_t* info, void* cuda_stream) {
  using namespace hpsi;
  if (!p || !psi || !eig_host) { set_error("null argument"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_davidson needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  hpsi_davidson_params_t prm = {1e-8, 200, 16, 1};
  if (params) prm = *params;
  if (prm.m_max < 2 || prm.m_max > MMAX || prm.max_iter < 1 || !(prm.tol >= 0.0)) { set_error("bad Davidson parameters"); return HPSI_EINVAL; }
  const int64_t n = p->sc.psi_len;
  if (n == 0) { set_error("empty target sector"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  // buffers: V[m][n] W[m][n] diag x wy r s | G[MMAX*MMAX] y[MMAX] c[MMAX] theta nrm[4] partial[MMAX*NB] counters[MMAX]
  const size_t small = MMAX * MMAX + 2 * MMAX + 8 + MMAX * NB + MMAX;
  const size_t need = (size_t)(2 * prm.m_max + 5) * n + small;
  if (p->dav_doubles < need) {
    cudaFree(p->d_dav);
    p->d_dav = nullptr;
    p->dav_doubles = 0;
    if (cudaMalloc(&p->d_dav, need * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      set_error("device allocation for the Davidson subspace failed");
      return HPSI_ENOMEM;
    }
    p->dav_doubles = need;
  }
  if (!p->h_dav) HPSI_CUDA(cudaMallocHost(&p->h_dav, 8 * sizeof(double)));
  double* V = p->d_dav;
  double* W = V + (size_t)prm.m_max * n;
  double* diag = W + (size_t)prm.m_max * n;
  double *x = diag + n, *wy = x + n, *r = wy + n, *s = r + n;
  double* G = s + n;
  double *y = G + MMAX * MMAX, *c = y + MMAX, *theta = c + MMAX, *nrm = theta + 1, *partial = nrm + 7;
  unsigned int* counters = reinterpret_cast<unsigned int*>(partial + MMAX * NB);
  HPSI_CUDA(cudaMemsetAsync(G, 0, small * sizeof(double), st));

  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* X, int nvec, const double* yv, double* out, int stride, double* mirror, int mstride) {
    dot_kernel<<<dim3(NB, nvec), 256, 0, st>>>(X, n, yv, n, partial, counters, out, stride, mirror, mstride);
  };
  int rc;
  if (prm.precondition && (rc = hpsi_diagonal(p, diag, cuda_stream)) != HPSI_OK) return rc;

  // V0 = psi/|psi| ; W0 = H V0
  dots(psi, 1, psi, nrm, 1, nullptr, 0);
  scale_kernel<<<eg, 256, 0, st>>>(V, psi, nullptr, nullptr, nrm, n);
  if ((rc = hpsi_apply(p, V, W, cuda_stream)) != HPSI_OK) return rc;
  int j = 1, nmv = 1, converged = 0;
  double rn = INFINITY, th = 0.0;
  for (int it = 0; it < prm.max_iter; ++it) {
    // new column of G = V^T W:  G[i][j-1] = G[j-1][i] = V_i . W_{j-1}
    dots(V, j, W + (size_t)(j - 1) * n, G + (j - 1), MMAX, G + (size_t)(j - 1) * MMAX, 1);
    small_eig_kernel<<<1, 32 * std::max(1, (j + 1) / 2), 0, st>>>(G, j, theta, y);
    ritz_kernel<<<eg, 256, 0, st>>>(V, W, n, j, y, theta, x, wy, r);
    dots(r, 1, r, nrm + 1, 1, nullptr, 0);                          // nrm[1] = |r|^2
    precond_kernel<<<eg, 256, 0, st>>>(r, diag, theta, prm.precondition, s, n);
    if (j >= prm.m_max) {                                           // restart with V = [x/|x|]
      dots(x, 1, x, nrm + 2, 1, nullptr, 0);
      scale_kernel<<<eg, 256, 0, st>>>(V, x, W, wy, nrm + 2, n);
      HPSI_CUDA(cudaMemsetAsync(G, 0, MMAX * MMAX * sizeof(double), st));
      set_scalar_kernel<<<1, 1, 0, st>>>(G, theta);
      j = 1;
    }
    for (int pass = 0; pass < 2; ++pass) {                          // classical Gram-Schmidt, twice
      dots(V, j, s, c, 1, nullptr, 0);
      project_kernel<<<eg, 256, 0, st>>>(s, V, n, j, c);
    }
    dots(s, 1, s, nrm + 3, 1, nullptr, 0);                          // nrm[3] = |s|^2
    scale_kernel<<<eg, 256, 0, st>>>(V + (size_t)j * n, s, nullptr, nullptr, nrm + 3, n);
    double* hostbuf = p->h_dav;
    HPSI_CUDA(cudaMemcpyAsync(hostbuf, theta, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaStreamSynchronize(st));
    th = hostbuf[0];
    rn = std::sqrt(hostbuf[2]);
    const double ns = std::sqrt(hostbuf[4]);
    if (rn <= prm.tol) { converged = 1; break; }
    if (!(ns >= 1e-14) || nmv >= prm.max_iter) break;
    if ((rc = hpsi_apply(p, V + (size_t)j * n, W + (size_t)j * n, cuda_stream)) != HPSI_OK) return rc;
    ++j;
    ++nmv;
  }
  // psi = x/|x|
  dots(x, 1, x, nrm + 2, 1, nullptr, 0);
  scale_kernel<<<eg, 256, 0, st>>>(psi, x, nullptr, nullptr, nrm + 2, n);
  HPSI_CUDA(cudaGetLastError());
  HPSI_CUDA(cudaStreamSynchronize(st));
  *eig_host = th;
  if (info) { info->n_matvec = nmv; info->converged = converged; info->residual = rn; }
  return HPSI_OK;
}

// ------------------------------------------------------------------------------------------------ Lanczos
// hpsi_lanczos: explicitly restarted Lanczos with full (CGS2) re-orthogonalisation, lowest eigenpair, single root -
// the other solver PAPER.md:62 names ("the Lanczos or Davidson method").  Same device buffers and kernels as
// hpsi_davidson; per iteration the host reads back theta, the last Ritz coefficient and |w|^2 to steer the loop
// (residual estimate beta_j |y_j|); the true residual |H x - theta x| is computed once at the end.
namespace {

// x = sum_i y_i V_i
__global__ void combine_kernel(const double* __restrict__ V, int64_t n, int j, const double* __restrict__ y, double* x) {
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int i = 0; i < j; ++i) s += y[i] * V[i * n + e];
    x[e] = s;
  }
}
// T[j][j] = alpha_j, T[j][j+1] = T[j+1][j] = beta_j = sqrt(|w|^2)   (T stored with leading dimension MMAX)
__global__ void lanczos_set_kernel(double* T, int j, const double* alpha, const double* beta2) {
  T[j * MMAX + j] = *alpha;
  if (j + 1 < MMAX) { const double b = sqrt(*beta2); T[j * MMAX + j + 1] = b; T[(j + 1) * MMAX + j] = b; }
}

}  // namespace

extern "C" int hpsi_lanczos(hpsi_plan_t* p, double* psi, double* eig_host, const hpsi_davidson_params_t* params,
                            hpsi_davidson_info_t* info, void* cuda_stream) {
  using namespace hpsi;
  if (!p || !psi || !eig_host) { set_error("null argument"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_lanczos needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  hpsi_davidson_params_t prm = {1e-8, 200, 16, 0};
  if (params) prm = *params;
  if (prm.m_max < 2 || prm.m_max > MMAX || prm.max_iter < 1 || !(prm.tol >= 0.0)) { set_error("bad Lanczos parameters"); return HPSI_EINVAL; }
  const int64_t n = p->sc.psi_len;
  if (n == 0) { set_error("empty target sector"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  // buffers: V[m][n] x w | T[MMAX*MMAX] y[MMAX] c[MMAX] c2[MMAX] theta nrm[7] partial[MMAX*NB] counters[MMAX]
  const size_t small = MMAX * MMAX + 3 * MMAX + 8 + MMAX * NB + MMAX;
  const size_t need = (size_t)(prm.m_max + 2) * n + small;
  if (p->dav_doubles < need) {
    cudaFree(p->d_dav);
    p->d_dav = nullptr;
    p->dav_doubles = 0;
    if (cudaMalloc(&p->d_dav, need * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      set_error("device allocation for the Lanczos basis failed");
      return HPSI_ENOMEM;
    }
    p->dav_doubles = need;
  }
  if (!p->h_dav) HPSI_CUDA(cudaMallocHost(&p->h_dav, 8 * sizeof(double)));
  double* V = p->d_dav;
  double* x = V + (size_t)prm.m_max * n;
  double* w = x + n;
  double* T = w + n;
  double *y = T + MMAX * MMAX, *c = y + MMAX, *c2 = c + MMAX, *theta = c2 + MMAX, *nrm = theta + 1, *partial = nrm + 7;
  unsigned int* counters = reinterpret_cast<unsigned int*>(partial + MMAX * NB);
  HPSI_CUDA(cudaMemsetAsync(T, 0, small * sizeof(double), st));
  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* X, int nvec, const double* yv, double* out) {
    dot_kernel<<<dim3(NB, nvec), 256, 0, st>>>(X, n, yv, n, partial, counters, out, 1, nullptr, 0);
  };
  int rc;
  dots(psi, 1, psi, nrm);
  scale_kernel<<<eg, 256, 0, st>>>(V, psi, nullptr, nullptr, nrm, n);
  int j = 0, nmv = 0, converged = 0;
  double th = 0.0;
  double* host = p->h_dav;
  for (;;) {
    if ((rc = hpsi_apply(p, V + (size_t)j * n, w, cuda_stream)) != HPSI_OK) return rc;
    ++nmv;
    dots(V, j + 1, w, c);                                            // c[j] = alpha_j
    project_kernel<<<eg, 256, 0, st>>>(w, V, n, j + 1, c);           // three-term recurrence + re-orthogonalisation
    dots(V, j + 1, w, c2);
    project_kernel<<<eg, 256, 0, st>>>(w, V, n, j + 1, c2);          // second Gram-Schmidt pass
    dots(w, 1, w, nrm + 3);                                          // beta_j^2
    lanczos_set_kernel<<<1, 1, 0, st>>>(T, j, c + j, nrm + 3);
    small_eig_kernel<<<1, 32 * std::max(1, (j + 2) / 2), 0, st>>>(T, j + 1, theta, y);
    HPSI_CUDA(cudaMemcpyAsync(host, theta, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaMemcpyAsync(host + 1, y + j, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaMemcpyAsync(host + 2, nrm + 3, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaStreamSynchronize(st));
    th = host[0];
    const double beta = std::sqrt(host[2]);
    const double est = beta * std::fabs(host[1]);
    const bool done = est <= prm.tol || !(beta >= 1e-14) || nmv >= prm.max_iter;
    if (done || j + 1 >= prm.m_max) {
      combine_kernel<<<eg, 256, 0, st>>>(V, n, j + 1, y, x);         // Ritz vector
      dots(x, 1, x, nrm + 2);
      if (done) break;
      scale_kernel<<<eg, 256, 0, st>>>(V, x, nullptr, nullptr, nrm + 2, n);   // restart from the Ritz vector
      HPSI_CUDA(cudaMemsetAsync(T, 0, MMAX * MMAX * sizeof(double), st));
      j = 0;
      continue;
    }
    scale_kernel<<<eg, 256, 0, st>>>(V + (size_t)(j + 1) * n, w, nullptr, nullptr, nrm + 3, n);
    ++j;
  }
  // psi = x/|x| ; true residual |H psi - theta psi|
  scale_kernel<<<eg, 256, 0, st>>>(psi, x, nullptr, nullptr, nrm + 2, n);
  if ((rc = hpsi_apply(p, psi, w, cuda_stream)) != HPSI_OK) return rc;
  ++nmv;
  set_scalar_kernel<<<1, 1, 0, st>>>(c, theta);
  project_kernel<<<eg, 256, 0, st>>>(w, psi, n, 1, c);
  dots(w, 1, w, nrm + 1);
  HPSI_CUDA(cudaMemcpyAsync(host, nrm + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
  HPSI_CUDA(cudaGetLastError());
  HPSI_CUDA(cudaStreamSynchronize(st));
  const double rn = std::sqrt(host[0]);
  converged = rn <= prm.tol * 10.0 || rn <= prm.tol;      // the estimate steered the loop; the true residual is reported
  *eig_host = th;
  if (info) { info->n_matvec = nmv; info->converged = converged; info->residual = rn; }
  return HPSI_OK;
}
