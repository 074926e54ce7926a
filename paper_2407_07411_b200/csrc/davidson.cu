// hpsi_davidson: Davidson-Liu, lowest eigenpair, single root (PAPER.md:62 names "Lanczos or Davidson"; the algorithm
// is DESIGN.md reading A21).  Every O(psi_length) operation and the small subspace eigenproblem (parallel Jacobi in one
// thread block) run on the device, five fused launches per iteration besides the mat-vec; the host reads back theta and
// the residual norm on a side stream while the orthogonalisation of the same iteration is still running, so the next
// mat-vec is enqueued without a bubble.  All reductions are two-stage with a fixed order: bitwise reproducible.
#include <algorithm>
#include <cmath>
#include <string>
#include <vector>

#include "plan_dev.h"

namespace {

using hpsi::launch_dependent;   // kernels.cuh: every kernel of this file starts with pdl_wait() and is launched as a dependent
using hpsi::pdl_wait;           // of the kernel before it in the stream (launch latency of ~9 boundaries per iteration)

constexpr int NB = 256;       // partial blocks per dot product
constexpr int MMAX = 32;

// out[v*stride] (and mirror[v*mstride] if given) = X_v . y for the nvec vectors X_v = X + v*ldx.
// Two stages in one launch: block (b, v) reduces its slice into partial[v][b]; the block that finishes last for vector v
// (ticket from an atomic counter - control only) adds the NB partials in a fixed order, so the result does not depend
// on which block that is and a run is bitwise reproducible.  The counter is left at zero for the next call.
__global__ void dot_kernel(const double* __restrict__ X, int64_t ldx, const double* __restrict__ y, int64_t n,
                           double* __restrict__ partial, unsigned int* __restrict__ counters, double* out, int stride,
                           double* mirror, int mstride) {
  pdl_wait();
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
                             int64_t n, const double* dead = nullptr) {
  pdl_wait();
  if (dead && *dead != 0.0) return;
  const double inv = 1.0 / sqrt(*nrm2);
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    dst[e] = src[e] * inv;
    if (dst2) dst2[e] = src2[e] * inv;
  }
}

__device__ __forceinline__ double warp_sum_d(double v);
__device__ __forceinline__ double warp_min_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_max_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Smallest eigenpair of the symmetric j x j matrix G (leading dimension MMAX) by parallel two-sided Jacobi, run by ONE
// thread block of nw = blockDim.x / 32 warps: the m/2 disjoint rotations of a round-robin round are applied together,
// pair k by warp k % nw, lane t = row t; first all column updates A J, then all row updates J^T (A J).  (A one-warp cyclic
// version took 86 us per call at j ~ 10 - a quarter of a Davidson iteration's fixed cost.)  Writes theta[0] and y[0..j);
// G is left untouched.  Shared memory is passed in so that the fused Gram kernel can run it in its last block.
struct EigSmem {
  double A[MMAX][MMAX + 1], Q[MMAX][MMAX + 1];
  double cs[MMAX / 2][2];
  double norms[2];
  // lowest_eig_warp: tridiagonal T (d, e), Householder scalars, work vectors, pivots of T - lo I and their reciprocals
  double d[MMAX], e[MMAX], beta[MMAX], v[MMAX], w[MMAX], l[MMAX], rq[MMAX], z[MMAX];
  int ok;
};
__device__ void small_eig_block(const double* __restrict__ G, int j, double* theta, double* y, EigSmem& sm, int k = 1) {
  const int t = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int m = (j + 1) & ~1;                            // players of the round-robin (a dummy one if j is odd)
  const int np = m > 1 ? m / 2 : 1;                      // pairs per round
  for (int c = wid; c < j; c += nw)
    if (t < j) { sm.A[t][c] = 0.5 * (G[t * MMAX + c] + G[c * MMAX + t]); sm.Q[t][c] = (t == c) ? 1.0 : 0.0; }
  __syncthreads();
  double prev_off = 0.0;
  for (int sweep = 0; sweep < 30 && j > 1; ++sweep) {
    if (wid == 0) {                                      // squared norms of the off-diagonal part and of the diagonal
      double off = 0.0, dg = 0.0;
      if (t < j) {
        dg = sm.A[t][t] * sm.A[t][t];
        for (int q = t + 1; q < j; ++q) off += sm.A[t][q] * sm.A[t][q];
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dg += __shfl_xor_sync(0xffffffffu, dg, o); }
      if (t == 0) { sm.norms[0] = off; sm.norms[1] = dg; }
    }
    __syncthreads();
    // Stop when the off-diagonal Frobenius norm is below 1e-15 of the matrix norm - the floor rounding leaves (every
    // rotation perturbs the entries by ~2^-53 of the norm) - or when a sweep no longer reduces it by at least 4x: Jacobi
    // converges quadratically, so stagnation means the floor has been reached.  (The first version asked for 1e-17, which
    // rounding never reaches: every call ran all 30 sweeps, 50-70 us at j ~ 12 - most of a Davidson iteration's overhead.)
    const double off = sm.norms[0], dg = sm.norms[1];
    if (off <= 1e-30 * (dg + 2.0 * off) || off < 1e-300 || (sweep > 0 && off > 0.0625 * prev_off && off <= 1e-26 * (dg + 2.0 * off))) break;
    prev_off = off;
    for (int r = 0; r < m - 1; ++r) {
      for (int k = wid; k < np; k += nw) {               // columns p, q of pair k (this pair's alone)
        int p, q;
        if (k == 0) { p = m - 1; q = r; }
        else { p = (r + k) % (m - 1); q = (r - k + m - 1) % (m - 1); }
        if (p > q) { const int tmp = p; p = q; q = tmp; }
        double c = 1.0, sn = 0.0;
        if (q < j) {                                     // not the dummy player
          const double apq = sm.A[p][q];
          if (fabs(apq) >= 1e-300) {
            // tan of the smaller rotation angle, t = sign(tau) / (|tau| + sqrt(1 + tau^2)) with tau = (aqq - app) / (2 apq),
            // written with one division, one square root and one reciprocal square root (the chain of three divisions and
            // two square roots was most of a round's latency, and the rounds are the critical path of the iteration)
            const double d = sm.A[q][q] - sm.A[p][p];
            const double tt = 2.0 * apq / (d + copysign(sqrt(d * d + 4.0 * apq * apq), d));
            c = rsqrt(1.0 + tt * tt);
            sn = tt * c;
          }
        }
        __syncwarp();
        if (t == 0) { sm.cs[k][0] = c; sm.cs[k][1] = sn; }
        if (sn != 0.0 && t < j) {
          const double akp = sm.A[t][p], akq = sm.A[t][q];
          sm.A[t][p] = c * akp - sn * akq;
          sm.A[t][q] = sn * akp + c * akq;
          const double qkp = sm.Q[t][p], qkq = sm.Q[t][q];
          sm.Q[t][p] = c * qkp - sn * qkq;
          sm.Q[t][q] = sn * qkp + c * qkq;
        }
      }
      __syncthreads();
      for (int k = wid; k < np; k += nw) {               // rows p, q
        int p, q;
        if (k == 0) { p = m - 1; q = r; }
        else { p = (r + k) % (m - 1); q = (r - k + m - 1) % (m - 1); }
        if (p > q) { const int tmp = p; p = q; q = tmp; }
        const double c = sm.cs[k][0], sn = sm.cs[k][1];
        if (sn != 0.0 && t < j) {
          const double apk = sm.A[p][t], aqk = sm.A[q][t];
          sm.A[p][t] = c * apk - sn * aqk;
          sm.A[q][t] = sn * apk + c * aqk;
        }
      }
      __syncthreads();
    }
  }
  __syncthreads();
  if (wid == 0) {                                        // the k lowest Ritz pairs, ascending: theta[r], y[r * MMAX + t]
    unsigned taken = 0u;
    for (int r = 0; r < k && r < j; ++r) {
      int best = -1;
      for (int i = 0; i < j; ++i)
        if (!((taken >> i) & 1u) && (best < 0 || sm.A[i][i] < sm.A[best][best])) best = i;
      taken |= 1u << best;
      if (t == 0) theta[r] = sm.A[best][best];
      if (t < j) y[r * MMAX + t] = sm.Q[t][best];
    }
  }
}
// Lowest eigenpair of the symmetric j x j matrix G (leading dimension MMAX) by ONE warp, lane t = row t, in the three
// classical steps of a selected-eigenpair solver:
//   1. Householder tridiagonalisation T = Z^T A Z (the reflector of step s stays in column s of the work matrix);
//   2. the lowest eigenvalue of T by multisection on the Sturm count: every lane counts the eigenvalues below its own
//      shift, so a round narrows the bracket 33x and 11-12 rounds reach 2^-53; the bracket's lower end `lo` has count 0;
//   3. inverse iteration with the shift lo: T - lo I is positive definite up to rounding, so its LDL^T factorisation (the
//      pivots q_i = d_i - lo - e_{i-1}^2 / q_{i-1}) needs no pivoting; two solves, Rayleigh quotient in T,
//      back-transformation y = Z x.
// Cost ~j (reflectors) + ~12 j divisions (counts) instead of 6-10 Jacobi sweeps of j rounds each: 5-10 us instead of
// 20-90 us at j = 4 .. 16 (measured per call inside dav_gram_eig_kernel) - the Jacobi solve was 60 % of the fixed
// cost of a Davidson iteration.  The result is checked (|A y - theta y| against the norm of A, NaN-safe); on failure the
// function returns false and the caller runs the Jacobi solver.  Writes theta[0], y[0 .. j).
__device__ bool lowest_eig_warp(const double* __restrict__ G, int j, double* theta, double* y, EigSmem& sm) {
  constexpr unsigned FULL = 0xffffffffu;
  constexpr double EPS = 1.1102230246251565e-16;
  const int t = threadIdx.x & 31;
  const bool in = t < j;
  for (int c = 0; c < j; ++c)
    if (in) { const double a = 0.5 * (G[t * MMAX + c] + G[c * MMAX + t]); sm.A[t][c] = a; sm.Q[t][c] = a; }
  __syncwarp();
  if (j == 1) {
    if (t == 0) { theta[0] = sm.A[0][0]; y[0] = 1.0; }
    return true;
  }
  // ---- 1. tridiagonalisation
  for (int s = 0; s + 2 < j; ++s) {
    const double xt = (in && t > s) ? sm.A[t][s] : 0.0;
    const double x0 = __shfl_sync(FULL, xt, s + 1);
    const double sig = warp_sum_d(t > s + 1 ? xt * xt : 0.0);
    if (sig == 0.0) {                                    // column already tridiagonal (the same on every lane)
      if (t == 0) { sm.e[s] = x0; sm.beta[s] = 0.0; }
      continue;
    }
    const double alpha = -copysign(sqrt(x0 * x0 + sig), x0);
    const double v1 = x0 - alpha;
    const double b = 2.0 / (sig + v1 * v1);
    const double vt = (t == s + 1) ? v1 : (t > s + 1 ? xt : 0.0);
    sm.v[t] = vt;
    __syncwarp();
    double pt = 0.0;
    if (in && t > s) {
      double p0 = 0.0, p1 = 0.0;                         // two chains: the loads of a pair overlap
      int u = s + 1;
      for (; u + 1 < j; u += 2) { p0 += sm.A[t][u] * sm.v[u]; p1 += sm.A[t][u + 1] * sm.v[u + 1]; }
      if (u < j) p0 += sm.A[t][u] * sm.v[u];
      pt = (p0 + p1) * b;
    }
    const double K = 0.5 * b * warp_sum_d(vt * pt);
    const double wt = pt - K * vt;
    sm.w[t] = wt;
    __syncwarp();
    if (in && t > s) {
#pragma unroll 4
      for (int u = s + 1; u < j; ++u) sm.A[t][u] -= vt * sm.w[u] + wt * sm.v[u];
      sm.A[t][s] = vt;                                   // the reflector, for the back-transformation
    }
    if (t == 0) { sm.e[s] = alpha; sm.beta[s] = b; }
    __syncwarp();
  }
  if (in) sm.d[t] = sm.A[t][t];
  if (t == 0) { sm.e[j - 2] = sm.A[j - 1][j - 2]; sm.e[j - 1] = 0.0; }
  __syncwarp();
  // ---- 2. lowest eigenvalue of T: bracket from Gershgorin discs and min(d), then multisection
  const double dt = in ? sm.d[t] : 0.0;
  const double rt = in ? (t > 0 ? fabs(sm.e[t - 1]) : 0.0) + (t + 1 < j ? fabs(sm.e[t]) : 0.0) : 0.0;
  const double tn = fmax(warp_max_d(fabs(dt) + rt), 1e-300);
  const double pivmin = fmax(EPS * EPS * tn, 1e-300);
  double lo = warp_min_d(in ? dt - rt : 1.7e308) - (2.0 * EPS * tn + pivmin);
  double hi = warp_min_d(in ? dt : 1.7e308) + (2.0 * EPS * tn + pivmin);
  // The counts run on the determinant form of the Sturm sequence, p_i = (d_i - x) p_{i-1} - e_{i-1}^2 p_{i-2} (sign
  // changes = negative pivots q_i = p_i / p_{i-1}): one FMA per step on the critical path instead of a division (~130 clk),
  // which made the counts 2/3 of this routine.  T is scaled by a power of two (exact) to norm [1, 2), so p cannot
  // overflow in 32 steps; it is re-scaled when it shrinks.
  const int ex = ilogb(tn);
  const double pm = scalbn(pivmin, -ex);
  if (in) {
    sm.v[t] = scalbn(dt, -ex);
    const double es = scalbn(t + 1 < j ? sm.e[t] : 0.0, -ex);
    sm.w[t] = es * es;
  }
  __syncwarp();
  lo = scalbn(lo, -ex);
  hi = scalbn(hi, -ex);
  for (int round = 0; round < 40; ++round) {
    const double x = lo + (hi - lo) * ((t + 1) * (1.0 / 33.0));
    // neg = "p_i is negative", an exact zero taking the sign opposite to p_{i-1} (the pivot form would make q_i = -pivmin);
    // the recurrence itself has no division, so a vanishing p_i needs no replacement: the only arithmetic on the critical
    // path is one FMA per step.  The magnitude is checked every fourth step (p changes by 2^-106 .. 2^3 per step).
    double pp = 1.0, p = sm.v[0] - x;
    bool neg = p <= 0.0;
    int cnt = neg;
    for (int i = 1; i < j; ++i) {
      const double pn = fma(sm.v[i] - x, p, -sm.w[i - 1] * pp);
      const bool nneg = pn < 0.0 || (pn == 0.0 && !neg);
      cnt += nneg != neg;
      neg = nneg;
      pp = p;
      p = pn;
      if ((i & 3) == 0) {
        const double mag = fmax(fabs(p), fabs(pp));
        if (mag < 1e-100) { p *= 0x1p400; pp *= 0x1p400; }
        else if (mag > 1e100) { p *= 0x1p-400; pp *= 0x1p-400; }
      }
    }
    // the first lane whose shift has an eigenvalue below it closes the bracket from above, the lane before it from below;
    // every lane recomputes those two shifts from the lane number (same expression, same bits: no shuffle needed)
    const unsigned below = __ballot_sync(FULL, cnt >= 1);
    const int l = below ? __ffs(below) - 1 : 32;
    const double nhi = l < 32 ? lo + (hi - lo) * ((l + 1) * (1.0 / 33.0)) : hi;
    const double nlo = l > 0 ? lo + (hi - lo) * (l * (1.0 / 33.0)) : lo;
    const bool conv = (nhi - nlo) <= 2.0 * EPS * fmax(fabs(nlo), fabs(nhi)) + 2.0 * pm || !(nlo > lo || nhi < hi);
    lo = nlo; hi = nhi;
    if (conv) break;
  }
  lo = scalbn(lo, ex);
  __syncwarp();
  // ---- 3. inverse iteration with the shift lo: pivots, multipliers, reciprocals.  count(lo) = 0 makes the pivots
  // positive up to rounding; the last one is ~(mu_1 - lo) times a factor that can reach 1e6, so it may come out as a small
  // NEGATIVE number: it is kept as it is (replacing it would put that much residual into the vector); only |q| < pivmin
  // is lifted.
  if (t == 0) {
    double q = sm.d[0] - lo;
    if (!(fabs(q) >= pivmin)) q = pivmin;
    for (int i = 0; i + 1 < j; ++i) {
      const double rq = 1.0 / q;
      const double li = sm.e[i] * rq;
      sm.rq[i] = rq;
      sm.l[i] = li;
      q = sm.d[i + 1] - lo - li * sm.e[i];
      if (!(fabs(q) >= pivmin)) q = pivmin;
    }
    sm.rq[j - 1] = 1.0 / q;
  }
  double yt = in ? 0.5 + ((t + 1) * 0.6180339887498949 - floor((t + 1) * 0.6180339887498949)) : 0.0;   // generic start vector
  for (int it = 0; it < 2; ++it) {
    sm.z[t] = yt;
    __syncwarp();
    if (t == 0) {                                        // L D L^T x = z: two first-order recurrences
      double zi = sm.z[0];
      for (int i = 0; i + 1 < j; ++i) { zi = sm.z[i + 1] - sm.l[i] * zi; sm.z[i + 1] = zi; }
      double xi = sm.z[j - 1] * sm.rq[j - 1];
      sm.z[j - 1] = xi;
      for (int i = j - 2; i >= 0; --i) { xi = sm.z[i] * sm.rq[i] - sm.l[i] * xi; sm.z[i] = xi; }
    }
    __syncwarp();
    yt = in ? sm.z[t] : 0.0;
    const double big = warp_max_d(fabs(yt));
    yt = big > 0.0 ? yt / big : yt;                      // against overflow of the squares
    const double nn = warp_sum_d(yt * yt);
    yt *= rsqrt(nn);
    __syncwarp();
  }
  // Rayleigh quotient in T
  sm.z[t] = yt;
  __syncwarp();
  double ty = 0.0;
  if (in) {
    ty = sm.d[t] * yt;
    if (t + 1 < j) ty += sm.e[t] * sm.z[t + 1];
    if (t > 0) ty += sm.e[t - 1] * sm.z[t - 1];
  }
  const double th = warp_sum_d(yt * ty);
  // y = Z x: the reflectors in reverse order
  for (int s = j - 3; s >= 0; --s) {
    const double b = sm.beta[s];
    if (b == 0.0) continue;
    const double vt = (in && t > s) ? sm.A[t][s] : 0.0;
    const double dot = warp_sum_d(vt * yt);
    yt -= b * dot * vt;
  }
  yt *= rsqrt(warp_sum_d(yt * yt));
  // check against the matrix itself (kept in sm.Q): max |A y - theta y| and the infinity norm of A
  __syncwarp();
  sm.z[t] = yt;
  __syncwarp();
  double ay = 0.0, an = 0.0;
  if (in)
    for (int u = 0; u < j; ++u) { const double a = sm.Q[t][u]; ay += a * sm.z[u]; an += fabs(a); }
  const double res = warp_max_d(in ? fabs(ay - th * yt) : 0.0);
  const double anorm = warp_max_d(an);
  const bool good = res <= 2e-13 * anorm + 1e-290 && th == th;      // NaN fails both comparisons
  if (good) {
    if (t == 0) theta[0] = th;
    if (in) y[t] = yt;
  }
  return good;
}

// One block: the lowest pair by lowest_eig_warp (warp 0), the Jacobi solver if k > 1 or if that result fails its check.
__device__ void small_eig_lowest_or_jacobi(const double* __restrict__ G, int j, double* theta, double* y, EigSmem& sm, int k) {
  if (k == 1) {
    if (threadIdx.x < 32) {
      const bool good = lowest_eig_warp(G, j, theta, y, sm);
      if (threadIdx.x == 0) sm.ok = good ? 1 : 0;
    }
    __syncthreads();
    if (sm.ok) return;
    __syncthreads();
  }
  small_eig_block(G, j, theta, y, sm, k);
}

__global__ void small_eig_kernel(const double* __restrict__ G, int j, double* theta, double* y, int k,
                                 int* fell_back = nullptr) {
  pdl_wait();
  __shared__ EigSmem sm;
  if (threadIdx.x == 0) sm.ok = 0;
  __syncthreads();
  small_eig_lowest_or_jacobi(G, j, theta, y, sm, k);
  if (fell_back && threadIdx.x == 0) *fell_back = (k == 1 && !sm.ok) ? 1 : 0;
}

// ---------------------------------------------------------------------------------- fused Davidson iteration kernels
// One Davidson iteration is five launches besides the mat-vec (it was twelve): every kernel below runs NB blocks, block b
// owning the slice [b * per, (b + 1) * per) of the vectors; phase A is element-wise on the slice, phase B takes the dot
// products the NEXT step needs on the same slice (warp w: dot products w, w + 8, ...), and the block that finishes last
// (ticket from an atomic counter - control only) adds the NB partials of every dot product in a fixed order.  `ctl[5]`
// != 0 ("dead": the correction vector vanished, |s| < 1e-14) turns the kernels that would overwrite results into no-ops,
// so the host may learn of it one iteration late.
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ bool dav_last_block(unsigned int* ticket) {
  __shared__ bool last;
  __syncthreads();
  if (threadIdx.x == 0) { __threadfence(); last = atomicAdd(ticket, 1u) == gridDim.x - 1; }
  __syncthreads();
  if (last) __threadfence();
  return last;
}
// sum of the NB partials of one dot product, by one warp, in a fixed order
__device__ __forceinline__ double dav_sum_partials(const double* partial, int lane) {
  const volatile double* pv = partial + lane * (NB / 32);
  double t = 0.0;
  for (int i = 0; i < NB / 32; ++i) t += pv[i];
  return warp_sum_d(t);
}
__device__ __forceinline__ void dav_slice(int64_t n, int64_t& lo, int64_t& hi) {
  const int64_t per = (n + NB - 1) / NB;
  lo = (int64_t)blockIdx.x * per;
  hi = lo + per < n ? lo + per : n;
  if (lo > hi) lo = hi;
}

// G[:, j-1] = G[j-1, :] = V^T W_{j-1};  then (last block) the smallest Ritz pair of G -> theta, y
__global__ void __launch_bounds__(256) dav_gram_eig_kernel(const double* __restrict__ V, const double* __restrict__ wl, int64_t n,
                                                           int j, double* partial, unsigned int* ticket, double* G,
                                                           double* theta, double* y, const double* ctl) {
  pdl_wait();
  __shared__ EigSmem sm;
  if (ctl[5] != 0.0) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int64_t lo, hi;
  dav_slice(n, lo, hi);
  for (int i = wid; i < j; i += nw) {
    const double* v = V + (int64_t)i * n;
    double s = 0.0;
    for (int64_t e = lo + lane; e < hi; e += 32) s += v[e] * wl[e];
    s = warp_sum_d(s);
    if (lane == 0) partial[i * NB + blockIdx.x] = s;
  }
  if (!dav_last_block(ticket)) return;
  for (int i = wid; i < j; i += nw) {
    const double t = dav_sum_partials(partial + i * NB, lane);
    if (lane == 0) { G[i * MMAX + (j - 1)] = t; G[(j - 1) * MMAX + i] = t; }
  }
  if (threadIdx.x == 0) *ticket = 0;
  __syncthreads();
  small_eig_lowest_or_jacobi(G, j, theta, y, sm, 1);
}

// x = V y, wy = W y, r = wy - theta x, s = r / (diag - theta) (or r);  c_i = V_i . s,  nrm_r2 = r . r
__global__ void __launch_bounds__(256) dav_ritz_kernel(const double* __restrict__ V, const double* __restrict__ W,
                                                       const double* __restrict__ diag, int64_t n, int j,
                                                       const double* __restrict__ y, const double* __restrict__ theta,
                                                       int precondition, double* x, double* wy, double* r, double* s,
                                                       double* partial, unsigned int* ticket, double* c, double* nrm_r2,
                                                       const double* ctl) {
  pdl_wait();
  if (ctl[5] != 0.0) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const double th = *theta;
  int64_t lo, hi;
  dav_slice(n, lo, hi);
  for (int64_t e = lo + threadIdx.x; e < hi; e += blockDim.x) {
    double sx = 0.0, sw = 0.0;
    for (int i = 0; i < j; ++i) { const double yi = y[i]; sx += yi * V[i * n + e]; sw += yi * W[i * n + e]; }
    const double rr = sw - th * sx;
    double v = rr;
    if (precondition) {
      double den = diag[e] - th;
      if (fabs(den) < 1e-8) den = (den < 0) ? -1e-8 : 1e-8;
      v /= den;
    }
    x[e] = sx; wy[e] = sw; r[e] = rr; s[e] = v;
  }
  __syncthreads();                                       // this block's slice of r and s is written (and visible to the block)
  for (int i = wid; i <= j; i += nw) {
    const double* a = i < j ? V + (int64_t)i * n : r;
    const double* b = i < j ? s : r;
    double t = 0.0;
    for (int64_t e = lo + lane; e < hi; e += 32) t += a[e] * b[e];
    t = warp_sum_d(t);
    if (lane == 0) partial[i * NB + blockIdx.x] = t;
  }
  if (!dav_last_block(ticket)) return;
  for (int i = wid; i <= j; i += nw) {
    const double t = dav_sum_partials(partial + i * NB, lane);
    if (lane == 0) { if (i < j) c[i] = t; else *nrm_r2 = t; }
  }
  if (threadIdx.x == 0) *ticket = 0;
}

// s -= sum_i c_in[i] V_i;  then either c_out[i] = V_i . s (first Gram-Schmidt pass) or nrm_s2 = s . s (second pass, which
// also raises the "dead" flag when |s| < 1e-14)
__global__ void __launch_bounds__(256) dav_project_kernel(double* s, const double* __restrict__ V, int64_t n, int j,
                                                          const double* __restrict__ c_in, double* partial,
                                                          unsigned int* ticket, double* c_out, double* nrm_s2, double* ctl,
                                                          double stamp) {
  pdl_wait();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int64_t lo, hi;
  dav_slice(n, lo, hi);
  for (int64_t e = lo + threadIdx.x; e < hi; e += blockDim.x) {
    double acc = s[e];
    for (int i = 0; i < j; ++i) acc -= c_in[i] * V[i * n + e];
    s[e] = acc;
  }
  __syncthreads();
  const int ndots = c_out ? j : 1;
  for (int i = wid; i < ndots; i += nw) {
    const double* a = c_out ? V + (int64_t)i * n : s;
    double t = 0.0;
    for (int64_t e = lo + lane; e < hi; e += 32) t += a[e] * s[e];
    t = warp_sum_d(t);
    if (lane == 0) partial[i * NB + blockIdx.x] = t;
  }
  if (!dav_last_block(ticket)) return;
  for (int i = wid; i < ndots; i += nw) {
    const double t = dav_sum_partials(partial + i * NB, lane);
    if (lane == 0) {
      if (c_out) c_out[i] = t;
      else { *nrm_s2 = t; if (!(t >= 1e-28) && ctl[5] == 0.0) ctl[5] = stamp; }
    }
  }
  if (threadIdx.x == 0) *ticket = 0;
}

// s -= sum_i c_i V_i
__global__ void project_kernel(double* s, const double* __restrict__ V, int64_t n, int j, const double* __restrict__ c) {
  pdl_wait();
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double acc = s[e];
    for (int i = 0; i < j; ++i) acc -= c[i] * V[i * n + e];
    s[e] = acc;
  }
}

__global__ void set_scalar_kernel(double* dst, const double* src) {
  pdl_wait();
  *dst = *src;
}

// restart: G = [[theta]] (a no-op while the dead flag is up, like the other kernels that change the subspace)
__global__ void reset_gram_kernel(double* G, const double* theta, const double* dead) {
  pdl_wait();
  if (*dead != 0.0) return;
  for (int i = threadIdx.x; i < MMAX * MMAX; i += blockDim.x) G[i] = i == 0 ? *theta : 0.0;
}

}  // namespace

// Test entry point (include/hpsi.h): the subspace eigensolver of the drivers on one host matrix.
extern "C" int hpsi_debug_small_eig(const double* g_host, int32_t j, int32_t k, double* theta_host, double* y_host,
                                    int32_t* fell_back_host) {
  using namespace hpsi;
  if (!g_host || !theta_host || !y_host || j < 1 || j > MMAX || k < 1 || k > j) { set_error("bad arguments"); return HPSI_EINVAL; }
  double* d = nullptr;
  HPSI_CUDA(cudaMalloc(&d, (2 * MMAX * MMAX + MMAX + 8) * sizeof(double)));
  std::vector<double> g(MMAX * MMAX, 0.0), yh(MMAX * MMAX, 0.0), th(MMAX, 0.0);
  for (int r = 0; r < j; ++r)
    for (int c = 0; c < j; ++c) g[r * MMAX + c] = g_host[r * j + c];
  double *dG = d, *dY = d + MMAX * MMAX, *dT = dY + MMAX * MMAX;
  int* dF = reinterpret_cast<int*>(dT + MMAX);
  cudaError_t e = cudaMemcpy(dG, g.data(), g.size() * sizeof(double), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    small_eig_kernel<<<1, 32 * std::min(8, std::max(1, (j + 1) / 2))>>>(dG, j, dT, dY, k, dF);
    e = cudaDeviceSynchronize();
  }
  int fb = 0;
  if (e == cudaSuccess) e = cudaMemcpy(yh.data(), dY, yh.size() * sizeof(double), cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(th.data(), dT, MMAX * sizeof(double), cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(&fb, dF, sizeof(int), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(e, "hpsi_debug_small_eig");
  for (int r = 0; r < k; ++r) {
    theta_host[r] = th[r];
    for (int c = 0; c < j; ++c) y_host[r * j + c] = yh[r * MMAX + c];
  }
  if (fell_back_host) *fell_back_host = fb;
  return HPSI_OK;
}

// hpsi_set_exchange hook: w (this rank's partial products of v, or partial diag(H) when v == nullptr) -> sum over ranks
static int exchange(hpsi_plan_t* p, const double* v, double* w, int64_t n, int nvec, int64_t ld, void* cuda_stream) {
  if (!p->exchange_fn) return HPSI_OK;
  const int rc = p->exchange_fn(p->exchange_user, v, w, n, nvec, ld, cuda_stream);
  if (rc != 0) {
    hpsi::set_error("the exchange callback (hpsi_set_exchange) failed with code " + std::to_string(rc));
    return HPSI_ESTATE;
  }
  return HPSI_OK;
}

extern "C" int hpsi_set_exchange(hpsi_plan_t* p, hpsi_exchange_fn fn, void* user) {
  if (!p) { hpsi::set_error("null plan"); return HPSI_EINVAL; }
  p->exchange_fn = fn;
  p->exchange_user = fn ? user : nullptr;
  return HPSI_OK;
}

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

  // buffers: V[m][n] W[m][n] diag x wy r s | G[MMAX*MMAX] y[MMAX] c[MMAX] c2[MMAX] theta ctl[7] partial[(MMAX+1)*NB] tickets
  const size_t small = MMAX * MMAX + 3 * MMAX + 8 + (MMAX + 1) * NB + MMAX;
  const size_t need = (size_t)(2 * prm.m_max + 5) * n + small;
  if (p->dav_doubles < need) {
    HPSI_CUDA(cudaStreamSynchronize(st));
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
  if (!p->dav_side) {
    HPSI_CUDA(cudaStreamCreateWithFlags(&p->dav_side, cudaStreamNonBlocking));
    for (auto& e : p->dav_ev) HPSI_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  double* V = p->d_dav;
  double* W = V + (size_t)prm.m_max * n;
  double* diag = W + (size_t)prm.m_max * n;
  double *x = diag + n, *wy = x + n, *r = wy + n, *s = r + n;
  double* G = s + n;
  double *y = G + MMAX * MMAX, *c = y + MMAX, *c2 = c + MMAX, *theta = c2 + MMAX, *ctl = theta + 1, *partial = ctl + 7;
  unsigned int* tickets = reinterpret_cast<unsigned int*>(partial + (MMAX + 1) * NB);
  // ctl: [0] |psi|^2  [1] |r|^2  [2] |x|^2  [3] |s|^2  [5] dead flag   (theta, ctl[0..5] are read back together)
  HPSI_CUDA(cudaMemsetAsync(G, 0, small * sizeof(double), st));

  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* X, int nvec, const double* yv, double* out, int stride, double* mirror, int mstride) {
    launch_dependent(dot_kernel, dim3(dim3(NB, nvec)), dim3(256), 0, st, X, n, yv, n, partial, tickets + 8, out, stride, mirror, mstride);
  };
  int rc;
  if (prm.precondition) {
    if ((rc = hpsi_diagonal(p, diag, cuda_stream)) != HPSI_OK) return rc;
    if ((rc = exchange(p, nullptr, diag, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
  }

  // V0 = psi/|psi| ; W0 = H V0   (the normalisation rides on the mat-vec's prep kernel)
  dots(psi, 1, psi, ctl, 1, nullptr, 0);
  if ((rc = apply_impl(p, psi, W, false, cuda_stream, ctl, V)) != HPSI_OK) return rc;
  if ((rc = exchange(p, V, W, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
  int j = 1, nmv = 1, converged = 0;
  int j_good = 1;                                        // columns of V / W that were valid when the last correction vector was built
  double rn = INFINITY, th = 0.0;
  double* hostbuf = p->h_dav;
  for (int it = 0; it < prm.max_iter; ++it) {
    // new column of G = V^T W and its smallest Ritz pair; Ritz vector, residual, correction vector and its overlaps with V
    launch_dependent(dav_gram_eig_kernel, dim3(NB), dim3(256), 0, st, V, W + (size_t)(j - 1) * n, n, j, partial, tickets, G, theta, y, ctl);
    launch_dependent(dav_ritz_kernel, dim3(NB), dim3(256), 0, st, V, W, diag, n, j, y, theta, prm.precondition, x, wy, r, s, partial, tickets + 1, c,
                                         ctl + 1, ctl);
    // theta and |r|^2 travel to the host on a side stream while the orthogonalisation below is still running.  With an
    // exchange hook (ranks in lockstep) the copy waits for the orthogonalisation: whether it sees this iteration's dead flag
    // must not depend on timing, or the ranks would issue different numbers of mat-vecs.
    auto read_back = [&]() -> int {
      HPSI_CUDA(cudaEventRecord(p->dav_ev[0], st));
      HPSI_CUDA(cudaStreamWaitEvent(p->dav_side, p->dav_ev[0], 0));
      HPSI_CUDA(cudaMemcpyAsync(hostbuf, theta, 7 * sizeof(double), cudaMemcpyDeviceToHost, p->dav_side));
      HPSI_CUDA(cudaEventRecord(p->dav_ev[1], p->dav_side));
      return HPSI_OK;
    };
    if (!p->exchange_fn && (rc = read_back()) != HPSI_OK) return rc;
    if (j >= prm.m_max) {                                           // restart with V = [x/|x|]
      dots(x, 1, x, ctl + 2, 1, nullptr, 0);
      launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, V, x, W, wy, ctl + 2, n, ctl + 5);
      launch_dependent(reset_gram_kernel, dim3(1), dim3(256), 0, st, G, theta, ctl + 5);
      j = 1;
      dots(V, 1, s, c, 1, nullptr, 0);
    }
    // classical Gram-Schmidt, twice; the second pass leaves |s|^2 (and the dead flag, stamped with the iteration)
    const double stamp = (double)(it + 1);
    launch_dependent(dav_project_kernel, dim3(NB), dim3(256), 0, st, s, V, n, j, c, partial, tickets + 2, c2, nullptr, ctl, stamp);
    launch_dependent(dav_project_kernel, dim3(NB), dim3(256), 0, st, s, V, n, j, c2, partial, tickets + 3, nullptr, ctl + 3, ctl, stamp);
    if (p->exchange_fn && (rc = read_back()) != HPSI_OK) return rc;
    HPSI_CUDA(cudaEventSynchronize(p->dav_ev[1]));
    th = hostbuf[0];
    rn = std::sqrt(hostbuf[2]);
    // theta, |r| are the last good ones whether or not the dead flag is up (a dead iteration's kernels are no-ops; the flag
    // of THIS iteration's correction can already be visible because the copy runs beside the orthogonalisation: an exact
    // eigenvector gives r = 0, hence s = 0): convergence is decided first
    if (rn <= prm.tol) { converged = 1; break; }
    const double dead = hostbuf[6];
    if (dead != 0.0) {
      // The correction vector vanished with |r| > tol.  A flag stamped by an earlier iteration was raised after that
      // iteration's read-back: the mat-vec enqueued for the dead vector and everything since were no-ops on the subspace,
      // so the host counters step back.
      if (dead != stamp) { j = j_good; --nmv; }
      // Unpreconditioned (s = r) that is a breakdown, and so is a vanished fallback vector (stamp + 0.5 below).
      // Preconditioned it means r/(diag - theta) lies in span(V) (H diagonal: it is the Ritz vector itself): reading A21c
      // retries with the residual itself.
      if (!prm.precondition || dead != std::floor(dead) || nmv >= prm.max_iter) break;
      HPSI_CUDA(cudaMemsetAsync(ctl + 5, 0, sizeof(double), st));
      HPSI_CUDA(cudaMemcpyAsync(s, r, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
      dots(V, j, s, c, 1, nullptr, 0);
      launch_dependent(dav_project_kernel, dim3(NB), dim3(256), 0, st, s, V, n, j, c, partial, tickets + 2, c2, nullptr, ctl, stamp + 0.5);
      launch_dependent(dav_project_kernel, dim3(NB), dim3(256), 0, st, s, V, n, j, c2, partial, tickets + 3, nullptr, ctl + 3, ctl, stamp + 0.5);
    } else if (nmv >= prm.max_iter) {
      break;
    }
    // V_j = s/|s| (written by the prep kernel), W_j = H V_j - enqueued while the orthogonalisation may still be running
    j_good = j;
    if ((rc = apply_impl(p, s, W + (size_t)j * n, false, cuda_stream, ctl + 3, V + (size_t)j * n)) != HPSI_OK) return rc;
    if ((rc = exchange(p, V + (size_t)j * n, W + (size_t)j * n, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
    ++j;
    ++nmv;
  }
  // psi = x/|x|
  dots(x, 1, x, ctl + 2, 1, nullptr, 0);
  launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, psi, x, nullptr, nullptr, ctl + 2, n, nullptr);
  HPSI_CUDA(cudaGetLastError());
  HPSI_CUDA(cudaStreamSynchronize(st));
  *eig_host = th;
  if (info) { info->n_matvec = nmv; info->converged = converged; info->residual = rn; }
  return HPSI_OK;
}

// ------------------------------------------------------------------------------------- block (multi-root) Davidson
// hpsi_davidson_multi: block Davidson-Liu for the k lowest eigenpairs (reading A21b; PAPER.md:62 names the
// method only).  The new correction vectors of an iteration are multiplied by H in ONE batched apply (hpsi_apply_multi
// when the plan was laid out for several vectors), so the operators stream from HBM once per iteration, not once per root.
namespace {

// x_r = V y_r, wy_r = W y_r, res_r = wy_r - theta_r x_r  for root r = blockIdx.y (y_r = Y + r * MMAX)
__global__ void ritz_multi_kernel(const double* __restrict__ V, const double* __restrict__ W, int64_t n, int j,
                                  const double* __restrict__ Y, const double* __restrict__ theta, double* X, double* WY,
                                  double* Rv) {
  pdl_wait();
  const int r = blockIdx.y;
  const double* y = Y + r * MMAX;
  const double th = theta[r];
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double sx = 0.0, sw = 0.0;
    for (int i = 0; i < j; ++i) { const double yi = y[i]; sx += yi * V[i * n + e]; sw += yi * W[i * n + e]; }
    X[r * n + e] = sx; WY[r * n + e] = sw; Rv[r * n + e] = sw - th * sx;
  }
}

// s = r / (diag - theta) with |den| clamped to >= 1e-8 keeping its sign; or s = r
__global__ void precond_kernel(const double* __restrict__ r, const double* __restrict__ diag,
                               const double* __restrict__ theta, int precondition, double* s, int64_t n) {
  pdl_wait();
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

__global__ void set_diag_kernel(double* G, const double* theta, int k) {
  pdl_wait();
  if ((int)threadIdx.x < k) G[threadIdx.x * MMAX + threadIdx.x] = theta[threadIdx.x];
}

}  // namespace

extern "C" int hpsi_davidson_multi(hpsi_plan_t* p, double* psi, int64_t ld, int32_t n_roots, double* eig_host,
                                   double* residual_host, const hpsi_davidson_params_t* params, hpsi_davidson_info_t* info,
                                   void* cuda_stream) {
  using namespace hpsi;
  if (!p || !psi || !eig_host) { set_error("null argument"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_davidson_multi needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  hpsi_davidson_params_t prm = {1e-8, 200, 16, 1};
  if (params) prm = *params;
  const int k = n_roots;
  if (prm.m_max < 2 || prm.m_max > MMAX || prm.max_iter < 1 || !(prm.tol >= 0.0)) { set_error("bad Davidson parameters"); return HPSI_EINVAL; }
  if (k < 1 || 2 * k > prm.m_max) { set_error("n_roots must be between 1 and m_max / 2"); return HPSI_EINVAL; }
  const int64_t n = p->sc.psi_len;
  if (n == 0) { set_error("empty target sector"); return HPSI_EINVAL; }
  if (ld < n) { set_error("vector stride below psi_length"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  // buffers: V[m][n] W[m][n] diag X[k][n] WY[k][n] R[k][n] s | G[MMAX^2] Y[MMAX^2] theta[MMAX] c[MMAX] nrm[MMAX] partial[MMAX*NB] counters
  const size_t small = 2 * MMAX * MMAX + 3 * MMAX + MMAX * NB + MMAX;
  const size_t need = (size_t)(2 * prm.m_max + 3 * k + 2) * n + small;
  if (p->dav_doubles < need) {
    HPSI_CUDA(cudaStreamSynchronize(st));
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
  std::vector<double> host(2 * MMAX + 2);
  double* V = p->d_dav;
  double* W = V + (size_t)prm.m_max * n;
  double* diag = W + (size_t)prm.m_max * n;
  double* X = diag + n;
  double* WY = X + (size_t)k * n;
  double* Rv = WY + (size_t)k * n;
  double* s = Rv + (size_t)k * n;
  double* G = s + n;
  double *Y = G + MMAX * MMAX, *theta = Y + MMAX * MMAX, *c = theta + MMAX, *nrm = c + MMAX, *partial = nrm + MMAX;
  unsigned int* counters = reinterpret_cast<unsigned int*>(partial + MMAX * NB);
  HPSI_CUDA(cudaMemsetAsync(G, 0, small * sizeof(double), st));
  const int eg = (int)std::min<int64_t>((n + 255) / 256, 2048);
  auto dots = [&](const double* Xv, int nvec, const double* yv, double* out, int stride, double* mirror, int mstride) {
    launch_dependent(dot_kernel, dim3(dim3(NB, nvec)), dim3(256), 0, st, Xv, n, yv, n, partial, counters, out, stride, mirror, mstride);
  };
  // W[j0 .. j0 + cnt) = H V[j0 .. j0 + cnt): as few passes over the operators as the plan's batch width allows
  auto apply_block = [&](int j0, int cnt) -> int {
    for (int off = 0; off < cnt; off += p->sc.nvec) {
      const int nb = std::min(p->sc.nvec, cnt - off);
      int rc = apply_impl(p, V + (size_t)(j0 + off) * n, W + (size_t)(j0 + off) * n, false, cuda_stream, nullptr, nullptr, nb, n, n);
      if (rc != HPSI_OK) return rc;
      if ((rc = exchange(p, V + (size_t)(j0 + off) * n, W + (size_t)(j0 + off) * n, n, nb, n, cuda_stream)) != HPSI_OK) return rc;
    }
    return HPSI_OK;
  };
  // s orthogonalised twice against V[0 .. j), normalised into V[j]; returns |s|^2 location nrm[slot]
  auto orth_append = [&](int j, int slot) {
    for (int pass = 0; pass < 2 && j > 0; ++pass) {
      dots(V, j, s, c, 1, nullptr, 0);
      launch_dependent(project_kernel, dim3(eg), dim3(256), 0, st, s, V, n, j, c);
    }
    dots(s, 1, s, nrm + slot, 1, nullptr, 0);
    launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, V + (size_t)j * n, s, nullptr, nullptr, nrm + slot, n, nullptr);
  };
  int rc;
  if (prm.precondition) {
    if ((rc = hpsi_diagonal(p, diag, cuda_stream)) != HPSI_OK) return rc;
    if ((rc = exchange(p, nullptr, diag, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
  }

  // start vectors, orthonormalised one after the other
  for (int i = 0; i < k; ++i) {
    HPSI_CUDA(cudaMemcpyAsync(s, psi + (size_t)i * ld, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
    orth_append(i, i);
  }
  if ((rc = apply_block(0, k)) != HPSI_OK) return rc;
  int j = k, g0 = 0, nmv = k, converged = 0;
  std::vector<double> th(k, 0.0), rn(k, INFINITY);
  for (;;) {
    for (int col = g0; col < j; ++col)                                // new columns (and rows) of G = V^T W
      dots(V, j, W + (size_t)col * n, G + col, MMAX, G + (size_t)col * MMAX, 1);
    g0 = j;
    launch_dependent(small_eig_kernel, dim3(1), dim3(32 * std::min(8, std::max(1, (j + 1) / 2))), 0, st, G, j, theta, Y, k, nullptr);
    launch_dependent(ritz_multi_kernel, dim3(dim3(eg, k)), dim3(256), 0, st, V, W, n, j, Y, theta, X, WY, Rv);
    for (int r = 0; r < k; ++r) dots(Rv + (size_t)r * n, 1, Rv + (size_t)r * n, nrm + r, 1, nullptr, 0);
    HPSI_CUDA(cudaMemcpyAsync(host.data(), theta, k * sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaMemcpyAsync(host.data() + MMAX, nrm, k * sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaStreamSynchronize(st));
    std::vector<int> todo;
    for (int r = 0; r < k; ++r) {
      th[r] = host[r];
      rn[r] = std::sqrt(host[MMAX + r]);
      if (rn[r] > prm.tol) todo.push_back(r);
    }
    if (todo.empty()) { converged = 1; break; }
    if (nmv >= prm.max_iter) break;
    if (j + (int)todo.size() > prm.m_max) {                           // restart from the Ritz vectors
      HPSI_CUDA(cudaMemcpyAsync(V, X, (size_t)k * n * sizeof(double), cudaMemcpyDeviceToDevice, st));
      HPSI_CUDA(cudaMemcpyAsync(W, WY, (size_t)k * n * sizeof(double), cudaMemcpyDeviceToDevice, st));
      HPSI_CUDA(cudaMemsetAsync(G, 0, MMAX * MMAX * sizeof(double), st));
      launch_dependent(set_diag_kernel, dim3(1), dim3(32), 0, st, G, theta, k);
      j = g0 = k;
    }
    // correction vectors of the unconverged roots, each orthogonalised against V and the ones appended before it.  Fast
    // path: all of them without a host round trip, their norms read back together; if one vanished (|s| < 1e-14, it
    // must be dropped and the later ones change) the iteration's appends are redone one by one.
    auto append_all = [&](bool check_each) -> int {
      int added = 0;
      for (int r : todo) {
        if (nmv + added >= prm.max_iter) break;
        launch_dependent(precond_kernel, dim3(eg), dim3(256), 0, st, Rv + (size_t)r * n, diag, theta + r, prm.precondition, s, n);
        orth_append(j + added, added);
        if (check_each) {
          cudaMemcpyAsync(host.data(), nrm + added, sizeof(double), cudaMemcpyDeviceToHost, st);
          cudaStreamSynchronize(st);
          if (!(host[0] >= 1e-28)) {
            if (!prm.precondition) continue;                          // dropped: the slot is reused by the next root
            // reading A21c: the preconditioned correction lies in span(V); retry with the residual itself
            launch_dependent(precond_kernel, dim3(eg), dim3(256), 0, st, Rv + (size_t)r * n, diag, theta + r, 0, s, n);
            orth_append(j + added, added);
            cudaMemcpyAsync(host.data(), nrm + added, sizeof(double), cudaMemcpyDeviceToHost, st);
            cudaStreamSynchronize(st);
            if (!(host[0] >= 1e-28)) continue;
          }
        }
        ++added;
      }
      return added;
    };
    int added = append_all(false);
    if (added > 0) {
      HPSI_CUDA(cudaMemcpyAsync(host.data(), nrm, added * sizeof(double), cudaMemcpyDeviceToHost, st));
      HPSI_CUDA(cudaStreamSynchronize(st));
      bool ok = true;
      for (int a = 0; a < added; ++a) ok = ok && host[a] >= 1e-28;
      if (!ok) added = append_all(true);
    }
    if (added == 0) break;
    if ((rc = apply_block(j, added)) != HPSI_OK) return rc;
    j += added;
    nmv += added;
  }
  for (int r = 0; r < k; ++r)
    HPSI_CUDA(cudaMemcpyAsync(psi + (size_t)r * ld, X + (size_t)r * n, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
  HPSI_CUDA(cudaGetLastError());
  HPSI_CUDA(cudaStreamSynchronize(st));
  double worst = 0.0;
  for (int r = 0; r < k; ++r) {
    eig_host[r] = th[r];
    if (residual_host) residual_host[r] = rn[r];
    worst = std::max(worst, rn[r]);
  }
  if (info) { info->n_matvec = nmv; info->converged = converged; info->residual = worst; }
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
  pdl_wait();
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int i = 0; i < j; ++i) s += y[i] * V[i * n + e];
    x[e] = s;
  }
}
// T[j][j] = alpha_j, T[j][j+1] = T[j+1][j] = beta_j = sqrt(|w|^2)   (T stored with leading dimension MMAX)
__global__ void lanczos_set_kernel(double* T, int j, const double* alpha, const double* beta2) {
  pdl_wait();
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
    launch_dependent(dot_kernel, dim3(dim3(NB, nvec)), dim3(256), 0, st, X, n, yv, n, partial, counters, out, 1, nullptr, 0);
  };
  int rc;
  dots(psi, 1, psi, nrm);
  launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, V, psi, nullptr, nullptr, nrm, n, nullptr);
  int j = 0, nmv = 0, converged = 0;
  double th = 0.0;
  double* host = p->h_dav;
  for (;;) {
    if ((rc = hpsi_apply(p, V + (size_t)j * n, w, cuda_stream)) != HPSI_OK) return rc;
    if ((rc = exchange(p, V + (size_t)j * n, w, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
    ++nmv;
    dots(V, j + 1, w, c);                                            // c[j] = alpha_j
    launch_dependent(project_kernel, dim3(eg), dim3(256), 0, st, w, V, n, j + 1, c);           // three-term recurrence + re-orthogonalisation
    dots(V, j + 1, w, c2);
    launch_dependent(project_kernel, dim3(eg), dim3(256), 0, st, w, V, n, j + 1, c2);          // second Gram-Schmidt pass
    dots(w, 1, w, nrm + 3);                                          // beta_j^2
    launch_dependent(lanczos_set_kernel, dim3(1), dim3(1), 0, st, T, j, c + j, nrm + 3);
    launch_dependent(small_eig_kernel, dim3(1), dim3(32 * std::max(1, (j + 2) / 2)), 0, st, T, j + 1, theta, y, 1, nullptr);
    HPSI_CUDA(cudaMemcpyAsync(host, theta, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaMemcpyAsync(host + 1, y + j, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaMemcpyAsync(host + 2, nrm + 3, sizeof(double), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaStreamSynchronize(st));
    th = host[0];
    const double beta = std::sqrt(host[2]);
    const double est = beta * std::fabs(host[1]);
    const bool done = est <= prm.tol || !(beta >= 1e-14) || nmv >= prm.max_iter;
    if (done || j + 1 >= prm.m_max) {
      launch_dependent(combine_kernel, dim3(eg), dim3(256), 0, st, V, n, j + 1, y, x);         // Ritz vector
      dots(x, 1, x, nrm + 2);
      if (done) break;
      launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, V, x, nullptr, nullptr, nrm + 2, n, nullptr);   // restart from the Ritz vector
      HPSI_CUDA(cudaMemsetAsync(T, 0, MMAX * MMAX * sizeof(double), st));
      j = 0;
      continue;
    }
    launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, V + (size_t)(j + 1) * n, w, nullptr, nullptr, nrm + 3, n, nullptr);
    ++j;
  }
  // psi = x/|x| ; true residual |H psi - theta psi|
  launch_dependent(scale_kernel, dim3(eg), dim3(256), 0, st, psi, x, nullptr, nullptr, nrm + 2, n, nullptr);
  if ((rc = hpsi_apply(p, psi, w, cuda_stream)) != HPSI_OK) return rc;
  if ((rc = exchange(p, psi, w, n, 1, n, cuda_stream)) != HPSI_OK) return rc;
  ++nmv;
  launch_dependent(set_scalar_kernel, dim3(1), dim3(1), 0, st, c, theta);
  launch_dependent(project_kernel, dim3(eg), dim3(256), 0, st, w, psi, n, 1, c);
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
