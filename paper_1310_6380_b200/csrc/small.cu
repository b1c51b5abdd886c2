// S6 for small matrices (n <= 112, e.g. the paper's M = 3 truncation: K is 98 x 98): the whole Hermitian matrix lives in
// shared memory (both triangles) and one CTA runs the unblocked Householder tridiagonalisation (zhetd2 form) on it; no
// global traffic and no launches between columns.  Larger matrices take the two-stage path (band.cu, bulge.cu): "one code
// path will not serve both".  Q^H A Q = T for the pencil of PAPER.md:94-104; DESIGN.md section 5.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int SNMAX = 112;
constexpr int ST = 256;

template <int K>
__device__ __forceinline__ void small_reduce(double (&v)[K], double *red, double *res) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < K; ++k) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
  }
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < K; ++k) red[warp * K + k] = v[k];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < K; ++k) {
      double x = 0.0;
      for (int w = 0; w < ST / 32; ++w) x += red[w * K + k];
      res[k] = x;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) v[k] = res[k];
}

__global__ void __launch_bounds__(ST) tridiag_small_kernel(int n, int lda, BatchRef A, double *d, double *e, int inner) {
  extern __shared__ __align__(16) unsigned char small_smem[];
  const int ld = n + 1;
  cplx *As = reinterpret_cast<cplx *>(small_smem);  // [n][ld], As[c * ld + r] = A(r, c), full Hermitian
  cplx *vs = As + (size_t)n * ld;                   // [SNMAX]
  cplx *ws = vs + SNMAX;                            // [SNMAX]
  cplx *ps = ws + SNMAX;                            // [2][SNMAX]
  double *red = reinterpret_cast<double *>(ps + 2 * SNMAX);  // [8][2]
  double *res = red + 16;                                    // [2]
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  const cplx *Ag = batch_ptr(A, cell, mi);
  double *dg = d + (size_t)z * n, *eg = e + (size_t)z * n;
  const int t = threadIdx.x, r = t & 127, g = t >> 7;

  for (int q = t; q < n * n; q += ST) {
    const int rr = q % n, cc = q / n;
    if (rr >= cc) {
      cplx x = Ag[(size_t)rr + (size_t)cc * lda];
      if (rr == cc) x.y = 0.0;
      As[cc * ld + rr] = x;
      if (rr > cc) As[rr * ld + cc] = cconj(x);
    }
  }
  __syncthreads();

  for (int j = 0; j + 1 < n; ++j) {
    const int base = j + 1, m = n - base;  // x = A[base:n, j], length m >= 1
    const cplx *xj = As + j * ld + base;
    double sv[1] = {0.0};
    for (int i = 1 + t; i < m; i += ST) sv[0] += xj[i].x * xj[i].x + xj[i].y * xj[i].y;
    small_reduce<1>(sv, red, res);
    const cplx al = xj[0];
    const double ss = sv[0];
    cplx tau, scale;
    double beta;
    if (ss == 0.0 && al.y == 0.0) {
      tau = cmake(0.0, 0.0); scale = cmake(0.0, 0.0); beta = al.x;
    } else {
      // norm and reciprocals without the IEEE square root and divisions (as in chase.cu: rsqrt / rcp.approx + Newton
      // steps, each good to about 1 ulp; tau, v and beta come from the same values, so H stays unitary to a few ulp)
      const double s2 = al.x * al.x + al.y * al.y + ss, inrm = rsqrt(s2);
      double nrm = s2 * inrm;
      nrm = fma(fma(-nrm, nrm, s2), 0.5 * inrm, nrm);
      beta = -copysign(nrm, al.x);
      const double ib = -copysign(inrm, al.x);
      tau = cmake((beta - al.x) * ib, -al.y * ib);
      const double dr = al.x - beta, di = al.y, dd = dr * dr + di * di;
      double den;
      asm("rcp.approx.ftz.f64 %0, %1;\n" : "=d"(den) : "d"(dd));
      den = fma(den, fma(-dd, den, 1.0), den);
      den = fma(den, fma(-dd, den, 1.0), den);
      scale = cmake(dr * den, -di * den);
    }
    if (t == 0) { dg[j] = As[j * ld + j].x; eg[j] = beta; }
    if (tau.x == 0.0 && tau.y == 0.0) continue;  // uniform: H = I
    if (t < m) vs[t] = (t == 0) ? cmake(1.0, 0.0) : cmul(xj[t], scale);
    __syncthreads();
    // p = tau A22 v: thread (r, g) sums the columns c = g, g + 2, ... of its row
    {
      // four independent partial sums: the row's dependent chain is m / 8 complex multiply-adds long instead of m / 2
      cplx acc = cmake(0.0, 0.0), acc1 = cmake(0.0, 0.0), acc2 = cmake(0.0, 0.0), acc3 = cmake(0.0, 0.0);
      if (r < m) {
        const cplx *row = As + (size_t)base * ld + base + r;
        int c = g;
        for (; c + 6 < m; c += 8) {
          cfma(acc, row[(size_t)c * ld], vs[c]);
          cfma(acc1, row[(size_t)(c + 2) * ld], vs[c + 2]);
          cfma(acc2, row[(size_t)(c + 4) * ld], vs[c + 4]);
          cfma(acc3, row[(size_t)(c + 6) * ld], vs[c + 6]);
        }
        for (; c < m; c += 2) cfma(acc, row[(size_t)c * ld], vs[c]);
        acc = cadd(cadd(acc, acc1), cadd(acc2, acc3));
      }
      if (r < SNMAX) ps[g * SNMAX + r] = acc;
    }
    __syncthreads();
    cplx p = cmake(0.0, 0.0), v = cmake(0.0, 0.0);
    if (r < m) { p = cmul(tau, cadd(ps[r], ps[SNMAX + r])); v = vs[r]; }
    double sd[2] = {0.0, 0.0};
    if (g == 0 && r < m) { sd[0] = p.x * v.x + p.y * v.y; sd[1] = p.x * v.y - p.y * v.x; }  // p^H v
    small_reduce<2>(sd, red, res);
    const cplx alpha = cmul(cmake(-0.5 * tau.x, -0.5 * tau.y), cmake(sd[0], sd[1]));
    cplx w = p;
    cfma(w, alpha, v);
    if (g == 0 && r < m) ws[r] = w;
    __syncthreads();
    // A22 <- A22 - v w^H - w v^H (both triangles)
    if (r < m) {
      for (int c = g; c < m; c += 2) {
        cplx a = As[(base + c) * ld + base + r];
        cfms(a, v, cconj(ws[c]));
        cfms(a, w, cconj(vs[c]));
        if (r == c) a.y = 0.0;
        As[(base + c) * ld + base + r] = a;
      }
    }
    __syncthreads();
  }
  if (t == 0) { dg[n - 1] = As[(n - 1) * ld + (n - 1)].x; eg[n - 1] = 0.0; }
}
}  // namespace

int tridiag_small_max_n() { return SNMAX; }

void launch_tridiag_small(int n, int lda, BatchRef A, double *d, double *e, int ncells, int inner, cudaStream_t s) {
  const size_t smem = ((size_t)n * (n + 1) + 4 * SNMAX) * sizeof(cplx) + 18 * sizeof(double);
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(tridiag_small_kernel, 215 * 1024, attr_mask);
  KScope ks(KC_TRIDIAG_SMALL, 16.0 * n * (double)n * n / 3.0 * ncells * inner, s);  // the 16 n^3 / 3 flops of S6
  tridiag_small_kernel<<<ncells * inner, ST, smem, s>>>(n, lda, A, d, e, inner);
}

}  // namespace bsk
