// S7: lowest nev eigenvalues of real symmetric tridiagonal matrices by Sturm-count multisection.
// count(x) = number of negative pivots of T - xI = number of eigenvalues < x (Sylvester); the k-th eigenvalue (0-based)
// is the infimum of { x : count(x) >= k+1 }.  Start interval: Gershgorin.  DESIGN.md section 5 (S7); lambda = omega^2 of
// PAPER.md:104.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int ST = 256;   // maximum threads per matrix (the launch uses 8 threads per wanted eigenvalue, rounded to warps)
constexpr int G = 8;      // interior shifts per eigenvalue per round -> the interval shrinks 9x per round
constexpr int ROUNDS = 24;   // 9^24 > 2^76

// Number of eigenvalues < x = number of negative q_i = p_i / p_{i-1}, q_0 = d_0 - x, q_i = d_i - x - e_{i-1}^2 / q_{i-1}
// (a zero pivot is replaced by a tiny negative one, the role of -pivmin in LAPACK dstebz).  Evaluated WITHOUT the division, whose latency (~100 cycles)
// would serialise the recurrence: p_i = (d_i - x) p_{i-1} - e_{i-1}^2 p_{i-2}, a sign change between p_{i-1} and p_i
// is a negative pivot.  The pair (p_{i-1}, p_i) is renormalised by the power of two that brings p_i into [1, 2) every
// FOURTH step (an exact scaling of both, which changes no ratio and no sign): the chain of a step is then one DFMA and the
// zero test, not DFMA -> exponent test -> multiply.  Between two renormalisations the pair may grow by ||T - x||^4 and
// shrink by (2^-52 ||T - x||)^4, far inside the exponent range for any matrix this path produces.
__device__ __forceinline__ void sturm_step(double di, double e2i, double x, double &p0, double &p1, int &cnt) {
  double p2 = fma(di - x, p1, -(e2i * p0));
  if (p2 == 0.0) p2 = -0x1p-200 * p1;  // q_i = -2^-200
  cnt += (p2 < 0.0) != (p1 < 0.0);
  p0 = p1;
  p1 = p2;
}
__device__ __forceinline__ void sturm_renorm(double &p0, double &p1) {
  const int ex = (__double2hiint(p1) >> 20) & 0x7ff;
  const double sc = __hiloint2double((2046 - ex) << 20, 0);  // 2^(1023 - ex): p1 -> [1, 2)
  p0 *= sc;
  p1 *= sc;
}
__device__ __forceinline__ int sturm_count(const double *__restrict__ d, const double *__restrict__ e2, int n, double x) {
  double p0 = 1.0, p1 = d[0] - x;
  if (p1 == 0.0) p1 = -0x1p-200;  // zero pivot -> tiny negative pivot (relative 2^-200: far below rounding)
  int cnt = p1 < 0.0;
  int i = 1;
  for (; i + 3 < n; i += 4) {
#pragma unroll
    for (int u = 0; u < 4; ++u) sturm_step(d[i + u], e2[i + u - 1], x, p0, p1, cnt);
    sturm_renorm(p0, p1);
  }
  for (; i < n; ++i) {
    sturm_step(d[i], e2[i - 1], x, p0, p1, cnt);
    sturm_renorm(p0, p1);
  }
  return cnt;
}

__global__ void __launch_bounds__(ST) sturm_kernel(int n, const double *__restrict__ dg, const double *__restrict__ eg,
                                                   int nev, double *__restrict__ lam, int root) {
  extern __shared__ double sm[];
  double *d = sm, *e2 = sm + n;
  __shared__ double s_lo, s_hi;
  __shared__ __align__(8) int cnts[ST];
  const int z = blockIdx.x, t = threadIdx.x;
  dg += (size_t)z * n;
  eg += (size_t)z * n;
  const int nthr = blockDim.x, EPB = nthr / G;  // eigenvalues per pass
  for (int i = t; i < n; i += nthr) {
    d[i] = dg[i];
    e2[i] = (i + 1 < n) ? eg[i] * eg[i] : 0.0;
  }
  __syncthreads();
  {
    // Gershgorin bounds: every thread takes rows t, t + nthr, ...; minimum and maximum over the CTA (exact, whatever the
    // order).  (One thread looping over all n rows, two square roots each, was a tenth of the kernel at n = 1922.)
    double lo = d[0], hi = d[0];
    for (int i = t; i < n; i += nthr) {
      const double l = i > 0 ? sqrt(e2[i - 1]) : 0.0, r = i + 1 < n ? sqrt(e2[i]) : 0.0;
      lo = fmin(lo, d[i] - l - r);
      hi = fmax(hi, d[i] + l + r);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
      hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    double *red = reinterpret_cast<double *>(cnts);  // (cnts is not in use yet: ST ints = ST / 2 doubles >= 2 per warp)
    if ((t & 31) == 0) { red[2 * (t >> 5)] = lo; red[2 * (t >> 5) + 1] = hi; }
    __syncthreads();
    if (t == 0) {
      for (int w = 1; w < (nthr + 31) / 32; ++w) { lo = fmin(lo, red[2 * w]); hi = fmax(hi, red[2 * w + 1]); }
      const double nrm = fmax(fabs(lo), fabs(hi));
      lo -= 2.0 * nrm * 2.3e-16 * n + 2.0 * 2.3e-308;
      hi += 2.0 * nrm * 2.3e-16 * n + 2.0 * 2.3e-308;
      s_lo = lo; s_hi = hi;
    }
  }
  __syncthreads();
  const int grp = t / G, sub = t % G;
  for (int k0 = 0; k0 < nev; k0 += EPB) {
    const int k = k0 + grp;  // eigenvalue index of this group
    double lo = s_lo, hi = s_hi;
    for (int round = 0; round < ROUNDS; ++round) {
      const double w = hi - lo;
      const double x = lo + w * ((double)(sub + 1) / (double)(G + 1));
      int c = 0;
      if (k < nev) c = sturm_count(d, e2, n, x);
      cnts[t] = c;
      __syncthreads();
      // new interval: [x_{m-1}, x_m] with m the first sub-shift whose count >= k+1  (x_{-1} = lo, x_G = hi)
      int m = G;
      for (int s2 = G - 1; s2 >= 0; --s2)
        if (cnts[grp * G + s2] >= k + 1) m = s2;
      const double nlo = m == 0 ? lo : lo + w * ((double)m / (double)(G + 1));
      const double nhi = m == G ? hi : lo + w * ((double)(m + 1) / (double)(G + 1));
      lo = nlo; hi = nhi;
      __syncthreads();
    }
    if (k < nev && sub == 0) {
      const double x = 0.5 * (lo + hi);
      lam[(size_t)z * nev + k] = root ? sqrt(fmax(x, 0.0)) : x;  // S8: omega = sqrt(max(lambda, 0)) if asked
    }
  }
}
}  // namespace

void launch_sturm(int n, const double *d, const double *e, int nev, double *lam, int nmat, cudaStream_t s, bool root) {
  const size_t smem = (size_t)2 * n * sizeof(double);
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(sturm_kernel, 200 * 1024, attr_mask);
  KScope ks(KC_STURM, 0.0, s);
  const int nthr = nev * G >= ST ? ST : ((nev * G + 31) / 32) * 32;  // few eigenvalues: small CTAs, more of them per SM
  sturm_kernel<<<nmat, nthr, smem, s>>>(n, d, e, nev, lam, root ? 1 : 0);
}

}  // namespace bsk
