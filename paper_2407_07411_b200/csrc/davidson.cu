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

// partial[v*NB + b] = sum over block b's slice of X_v[e] * y[e]
__global__ void dot_partial_kernel(const double* __restrict__ X, int64_t ldx, const double* __restrict__ y, int64_t n,
                                   double* __restrict__ partial) {
  __shared__ double red[256];
  const double* x = X + (int64_t)blockIdx.y * ldx;
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
  if (threadIdx.x == 0) partial[blockIdx.y * NB + blockIdx.x] = red[0];
}
// out[v*stride] (and mirror[v*mstride] if given) = sum_b partial[v][b], b ascending
__global__ void dot_final_kernel(const double* __restrict__ partial, int nvec, double* out, int stride, double* mirror,
                                 int mstride) {
  const int v = threadIdx.x;
  if (v >= nvec) return;
  double s = 0.0;
  for (int b = 0; b < NB; ++b) s += partial[v * NB + b];
  out[(int64_t)v * stride] = s;
  if (mirror) mirror[(int64_t)v * mstride] = s;
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

// Smallest eigenpair of the symmetric j x j matrix G (leading dimension MMAX) by cyclic Jacobi, one warp.
// Writes theta[0] and y[0..j).  G itself is left untouched (work copy in shared memory).
__global__ void small_eig_kernel(const double* __restrict__ G, int j, double* theta, double* y) {
  __shared__ double A[MMAX][MMAX + 1], Q[MMAX][MMAX + 1];
  const int t = threadIdx.x;
  for (int c = 0; c < j; ++c)
    if (t < j) { A[t][c] = 0.5 * (G[t * MMAX + c] + G[c * MMAX + t]); Q[t][c] = (t == c) ? 1.0 : 0.0; }
  __syncwarp();
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0, dg = 0.0;
    for (int p = 0; p < j; ++p) {
      dg += A[p][p] * A[p][p];
      for (int q = p + 1; q < j; ++q) off += A[p][q] * A[p][q];
    }
    if (off <= 1e-34 * (dg + 2.0 * off) || off < 1e-300) break;   // off-diagonal norm below 1e-17 of the matrix norm
    for (int p = 0; p < j - 1; ++p)
      for (int q = p + 1; q < j; ++q) {
        const double apq = A[p][q];
        if (fabs(apq) < 1e-300) continue;                 // uniform: every lane reads the same value
        const double app = A[p][p], aqq = A[q][q];
        const double tau = (aqq - app) / (2.0 * apq);
        const double tt = (tau >= 0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
        const double c = 1.0 / sqrt(1.0 + tt * tt), s = tt * c;
        __syncwarp();
        if (t < j) {                                      // columns p,q
          const double akp = A[t][p], akq = A[t][q];
          A[t][p] = c * akp - s * akq;
          A[t][q] = s * akp + c * akq;
          const double qkp = Q[t][p], qkq = Q[t][q];
          Q[t][p] = c * qkp - s * qkq;
          Q[t][q] = s * qkp + c * qkq;
        }
        __syncwarp();
        if (t < j) {                                      // rows p,q
          const double apk = A[p][t], aqk = A[q][t];
          A[p][t] = c * apk - s * aqk;
          A[q][t] = s * apk + c * aqk;
        }
        __syncwarp();
      }
  }
  __syncwarp();
  int best = 0;
  for (int i = 1; i < j; ++i)
    if (A[i][i] < A[best][best]) best = i;
  if (t == 0) theta[0] = A[best][best];
  if (t < j) y[t] = Q[t][best];
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

  // buffers: V[m][n] W[m][n] diag x wy r s | G[MMAX*MMAX] y[MMAX] c[MMAX] theta nrm[4] partial[MMAX*NB]
  const size_t small = MMAX * MMAX + 2 * MMAX + 8 + MMAX * NB;
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
  HPSI_CUDA(cudaMemsetAsync(G, 0, small * sizeof(double), st));

  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* X, int nvec, const double* yv, double* out, int stride, double* mirror, int mstride) {
    dot_partial_kernel<<<dim3(NB, nvec), 256, 0, st>>>(X, n, yv, n, partial);
    dot_final_kernel<<<1, MMAX, 0, st>>>(partial, nvec, out, stride, mirror, mstride);
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
    small_eig_kernel<<<1, 32, 0, st>>>(G, j, theta, y);
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

  // buffers: V[m][n] x w | T[MMAX*MMAX] y[MMAX] c[MMAX] c2[MMAX] theta nrm[7] partial[MMAX*NB]
  const size_t small = MMAX * MMAX + 3 * MMAX + 8 + MMAX * NB;
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
  HPSI_CUDA(cudaMemsetAsync(T, 0, small * sizeof(double), st));
  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* X, int nvec, const double* yv, double* out) {
    dot_partial_kernel<<<dim3(NB, nvec), 256, 0, st>>>(X, n, yv, n, partial);
    dot_final_kernel<<<1, MMAX, 0, st>>>(partial, nvec, out, 1, nullptr, 0);
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
    small_eig_kernel<<<1, 32, 0, st>>>(T, j + 1, theta, y);
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
