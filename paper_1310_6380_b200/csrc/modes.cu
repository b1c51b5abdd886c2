// Mode shapes ("the eigenvectors U give the displacement mode shapes and
// S = -Phi^-1 H* U the stress mode shapes").  Route: the Hermitian BAND matrix of S6 stage 1 is kept; for every wanted
// eigenvalue (from the Sturm bisection of S7) its eigenvector is found by inverse iteration on the band matrix (pivoted band
// LU, one CTA per k-point, a sliding window of b + 1 rows in shared memory); the vectors then go back through the block
// reflectors of stage 1 (GEMMs, api.cu), through L_Psi^-H, and S = Phi^-1 H U.  Stage 2 (the bulge chase) is not involved.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int MT = 128;  // threads per CTA

__device__ __forceinline__ double cabs2(cplx a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ cplx crcp(cplx a) {
  const double d = 1.0 / (a.x * a.x + a.y * a.y);
  return cmake(a.x * d, -a.y * d);
}
// B[r, c] of the Hermitian band matrix (lower storage ab[c * ld + (r - c)], 0 <= r - c <= b), zero outside the band
__device__ __forceinline__ cplx band_at(const cplx *__restrict__ ab, int ld, int b, int n, int r, int c) {
  if (c < 0 || c >= n || r < 0 || r >= n) return cmake(0.0, 0.0);
  if (r >= c) return r - c <= b ? ab[(size_t)c * ld + (r - c)] : cmake(0.0, 0.0);
  return c - r <= b ? cconj(ab[(size_t)r * ld + (c - r)]) : cmake(0.0, 0.0);
}
__device__ __forceinline__ double block_sum(double v, double *red) {  // every thread gets the same bits
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double s = 0.0;
  for (int w = 0; w < MT / 32; ++w) s += red[w];
  return s;
}

// One CTA per matrix (k-point).  For j = 0 .. nvec-1: shift sigma_j next to lam[j], LU = P (B - sigma_j I) with partial
// pivoting (L: b multipliers per column, U: 2b + 1 entries per row, written to `lu`), three steps of inverse iteration from
// a fixed start vector, each followed by modified Gram-Schmidt against the earlier vectors whose eigenvalue lies within
// `ortol` (LAPACK zstein's criterion: 1e-3 of the matrix norm), and normalisation.  Z: n x nvec per matrix (ld n).
// lu per matrix: n (2b + 1) [U rows] + n b [L] complex, then n ints [pivots] (in the space of n / 4 + 1 more complex).
__global__ void __launch_bounds__(MT) band_invit_kernel(int n, int b, int ld, BatchRef AB, const double *__restrict__ lam_all,
                                                        int nvec, BatchRef Zr, BatchRef LUr, int inner) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = 2 * b + 2, R = b + 1;
  cplx *win = reinterpret_cast<cplx *>(smem_raw);        // [R][W]
  cplx *x = win + (size_t)R * W;                          // [n]
  double *red = reinterpret_cast<double *>(x + n);        // [MT / 32]
  int *s_piv = reinterpret_cast<int *>(red + MT / 32);
  const int z = blockIdx.x, cell = z / inner, mi = z % inner, t = threadIdx.x;
  const cplx *ab = batch_ptr(AB, cell, mi);
  cplx *Z = batch_ptr(Zr, cell, mi);
  cplx *Urow = batch_ptr(LUr, cell, mi);
  cplx *Lmul = Urow + (size_t)n * (2 * b + 1);
  int *piv = reinterpret_cast<int *>(Lmul + (size_t)n * b);
  const double *lam = lam_all + (size_t)z * nvec;

  // scale of the matrix: the largest absolute row sum (infinity norm)
  double nrm = 0.0;
  for (int r = t; r < n; r += MT) {
    double s = 0.0;
    for (int c = r - b; c <= r + b; ++c) s += sqrt(cabs2(band_at(ab, ld, b, n, r, c)));
    nrm = fmax(nrm, s);
  }
  {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm = fmax(nrm, __shfl_xor_sync(0xffffffffu, nrm, o));
    if ((t & 31) == 0) red[t >> 5] = nrm;
    __syncthreads();
    nrm = 0.0;
    for (int w = 0; w < MT / 32; ++w) nrm = fmax(nrm, red[w]);
    __syncthreads();
  }
  const double eps = 2.220446049250313e-16, tiny = eps * fmax(nrm, 1e-300), ortol = 1e-3 * nrm;
  double sigma_prev = 0.0;

  for (int j = 0; j < nvec; ++j) {
    // shift: a hair off the computed eigenvalue; equal eigenvalues get distinct shifts (zstein)
    double sigma = lam[j] - 2.0 * tiny;
    if (j > 0 && sigma <= sigma_prev + 8.0 * tiny) sigma = sigma_prev + 10.0 * tiny;
    sigma_prev = sigma;
    // ---------------------------------------------------------------- factorisation, rows i .. i + b in the window
    for (int q = t; q < R * W; q += MT) {
      const int r = q / W, cs = q % W;                      // window row r (slot r), column slot cs = column cs
      cplx v = band_at(ab, ld, b, n, r, cs);
      if (r == cs) v.x -= sigma;
      if (r >= n || cs > 2 * b) v = cmake(0.0, 0.0);         // (column 2b + 1 enters with row b + 1)
      win[q] = v;
    }
    __syncthreads();
    for (int i = 0; i < n; ++i) {
      const int nrows = min(b, n - 1 - i), ci = i % W, si = i % R;
      if (t == 0) {  // partial pivoting: first row of largest modulus in column i
        int best = i;
        double bv = cabs2(win[si * W + ci]);
        for (int r = i + 1; r <= i + nrows; ++r) {
          const double v = cabs2(win[(r % R) * W + ci]);
          if (v > bv) { bv = v; best = r; }
        }
        *s_piv = best;
        piv[i] = best;
      }
      __syncthreads();
      const int pr = *s_piv, sp = pr % R;
      if (pr != i)
        for (int c = t; c < W; c += MT) {
          const cplx a = win[si * W + c];
          win[si * W + c] = win[sp * W + c];
          win[sp * W + c] = a;
        }
      __syncthreads();
      cplx pivot = win[si * W + ci];
      if (cabs2(pivot) < tiny * tiny) pivot = cmake(tiny, 0.0);   // exactly singular: perturb (the role of zlagtf's tol)
      const cplx rp = crcp(pivot);
      for (int c = t; c <= 2 * b; c += MT) Urow[(size_t)i * (2 * b + 1) + c] = c == 0 ? pivot : win[si * W + (i + c) % W];
      for (int q = t; q < nrows * (2 * b + 1); q += MT) {
        const int r = i + 1 + q / (2 * b + 1), c = q % (2 * b + 1), sr = r % R;
        const cplx m = cmul(win[sr * W + ci], rp);
        if (c == 0) Lmul[(size_t)i * b + (r - i - 1)] = m;
        else {
          cplx a = win[sr * W + (i + c) % W];
          cfms(a, m, win[si * W + (i + c) % W]);
          win[sr * W + (i + c) % W] = a;
        }
      }
      __syncthreads();
      // the window moves on: column i leaves (its slot will hold column i + W), row i + b + 1 enters into the slot of row i
      for (int r = 1 + t; r <= nrows; r += MT) win[((i + r) % R) * W + ci] = cmake(0.0, 0.0);
      const int rn = i + b + 1;
      if (rn < n) {
        for (int c = t; c < W; c += MT) {
          const int col = i + 1 + c;                         // columns i + 1 .. i + 2b + 2
          cplx v = band_at(ab, ld, b, n, rn, col);
          if (col == rn) v.x -= sigma;
          win[si * W + col % W] = v;
        }
      }
      __syncthreads();
    }
    // ---------------------------------------------------------------- inverse iteration
    for (int r = t; r < n; r += MT) {  // fixed start vector (a different one per j)
      const unsigned h = (unsigned)(r * 2654435761u) ^ (unsigned)((j + 1) * 40503u);
      x[r] = cmake(1.0 + (double)(h & 1023) / 1024.0, (double)((h >> 10) & 1023) / 1024.0 - 0.5);
    }
    __syncthreads();
    for (int it = 0; it < 3; ++it) {
      if (t < 32) {
        // forward: row interchanges and the multipliers of L, one column at a time; lane r owns row i + 1 + r
        for (int i = 0; i < n; ++i) {
          const int nrows = min(b, n - 1 - i), pr = piv[i];
          if (t == 0 && pr != i) { const cplx a = x[i]; x[i] = x[pr]; x[pr] = a; }
          __syncwarp();
          const cplx xi = x[i];
          if (t < nrows) { cplx a = x[i + 1 + t]; cfms(a, Lmul[(size_t)i * b + t], xi); x[i + 1 + t] = a; }
          __syncwarp();
        }
        // backward, column oriented: x[i] = x[i] / U[i,i], then x[i - c] -= U[i - c, i] x[i], c = 1 .. 2b
        for (int i = n - 1; i >= 0; --i) {
          cplx xi = cmake(0.0, 0.0);
          if (t == 0) { xi = cmul(x[i], crcp(Urow[(size_t)i * (2 * b + 1)])); x[i] = xi; }
          xi = cmake(__shfl_sync(0xffffffffu, xi.x, 0), __shfl_sync(0xffffffffu, xi.y, 0));
          for (int c = 1 + t; c <= 2 * b; c += 32) {
            const int r = i - c;
            if (r >= 0) { cplx a = x[r]; cfms(a, Urow[(size_t)r * (2 * b + 1) + c], xi); x[r] = a; }
          }
          __syncwarp();
        }
      }
      __syncthreads();
      // modified Gram-Schmidt against the earlier vectors of the cluster, then normalisation
      for (int p = 0; p < j; ++p) {
        if (fabs(lam[j] - lam[p]) > ortol) continue;
        const cplx *zp = Z + (size_t)p * n;
        double dr = 0.0, di = 0.0;
        for (int r = t; r < n; r += MT) { const cplx a = zp[r], c2 = x[r]; dr += a.x * c2.x + a.y * c2.y; di += a.x * c2.y - a.y * c2.x; }
        dr = block_sum(dr, red);
        di = block_sum(di, red);
        for (int r = t; r < n; r += MT) { cplx c2 = x[r]; cfms(c2, zp[r], cmake(dr, di)); x[r] = c2; }
        __syncthreads();
      }
      double s = 0.0;
      for (int r = t; r < n; r += MT) s += cabs2(x[r]);
      s = block_sum(s, red);
      const double inv = 1.0 / sqrt(s);
      for (int r = t; r < n; r += MT) x[r] = cscale(x[r], inv);
      __syncthreads();
    }
    for (int r = t; r < n; r += MT) Z[(size_t)j * n + r] = x[r];
    __syncthreads();
  }
}

// HU = V B(k) U on the N plane waves of every mode (eq. 18; H = V B, B = i (k + G) on diagonal blocks):
// rows (1,g) = i V kx_g U1[g], (2,g) = i V ky_g U2[g], (3,g) = i V (ky_g U1[g] + kx_g U2[g]).
__global__ void __launch_bounds__(256) apply_h_kernel(int N, double V, BatchRef U, int ldu, BatchRef HU, int ldh, BatchRef KAP,
                                                      int nvec, int inner) {
  const int z = blockIdx.z, cell = z / inner, mi = z % inner;
  const int g = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (g >= N || j >= nvec) return;
  const cplx *u = batch_ptr(U, cell, mi) + (size_t)j * ldu;
  cplx *h = batch_ptr(HU, cell, mi) + (size_t)j * ldh;
  const double *kap = reinterpret_cast<const double *>(batch_ptr(KAP, cell, mi));  // [x | y][N] doubles of this k-point
  const double kx = kap[g], ky = kap[N + g];
  const cplx u1 = u[g], u2 = u[N + g];
  // i * (a + i b) = -b + i a
  h[g] = cmake(-V * kx * u1.y, V * kx * u1.x);
  h[N + g] = cmake(-V * ky * u2.y, V * ky * u2.x);
  h[2 * N + g] = cmake(-V * (ky * u1.y + kx * u2.y), V * (ky * u1.x + kx * u2.x));
}

// Rayleigh quotients in factored form: omega^2_j = (H u_j)^dagger (Phi^-1 H u_j) / (y_j^dagger y_j), u = L_Psi^-H y.
// For omega^2 << lambda_max this is far more accurate than the eigenvalue of the assembled pencil (whose absolute error
// is ~eps lambda_max): the quotient is second-order accurate in the vector and every factor is computed to a relative
// error of ~eps kappa(Phi) (the singular-value route of SURVEY 8(c)-7 / reading R8, reached without an SVD).
__global__ void __launch_bounds__(256) rayleigh_kernel(int n3, int n2, BatchRef HU, BatchRef S, int lds, BatchRef Y, int ldy,
                                                       double *__restrict__ out, int nvec, int inner) {
  __shared__ double red[2][8];
  const int z = blockIdx.y, cell = z / inner, mi = z % inner, j = blockIdx.x;
  const cplx *h = batch_ptr(HU, cell, mi) + (size_t)j * lds, *sv = batch_ptr(S, cell, mi) + (size_t)j * lds;
  const cplx *y = batch_ptr(Y, cell, mi) + (size_t)j * ldy;
  double num = 0.0, den = 0.0;
  for (int i = threadIdx.x; i < n3; i += 256) num += h[i].x * sv[i].x + h[i].y * sv[i].y;  // Re conj(h) s
  for (int i = threadIdx.x; i < n2; i += 256) den += y[i].x * y[i].x + y[i].y * y[i].y;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    num += __shfl_xor_sync(0xffffffffu, num, o);
    den += __shfl_xor_sync(0xffffffffu, den, o);
  }
  if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = num; red[1][threadIdx.x >> 5] = den; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) { a += red[0][w]; b += red[1][w]; }
    out[(size_t)z * nvec + j] = a / b;
  }
}
}  // namespace

size_t band_invit_lu_elems(int n, int b) { return (size_t)n * (2 * b + 1) + (size_t)n * b + (size_t)n / 4 + 16; }

void launch_band_invit(int n, int b, BatchRef AB, const double *lam, int nvec, BatchRef Z, BatchRef LU, int ncells, int inner,
                       cudaStream_t s) {
  const size_t smem = ((size_t)(b + 1) * (2 * b + 2) + n) * sizeof(cplx) + (MT / 32) * sizeof(double) + 16;
  static unsigned long long mask = 0;
  ensure_dyn_smem(band_invit_kernel, 100 * 1024, mask);
  KScope ks(KC_OTHER, 0.0, s);
  band_invit_kernel<<<ncells * inner, MT, smem, s>>>(n, b, 2 * b, AB, lam, nvec, Z, LU, inner);
}

void launch_apply_h(int N, double V, BatchRef U, int ldu, BatchRef HU, int ldh, BatchRef KAP, int nvec, int ncells,
                    int inner, cudaStream_t s) {
  KScope ks(KC_OTHER, 0.0, s);
  apply_h_kernel<<<dim3((N + 255) / 256, nvec, ncells * inner), 256, 0, s>>>(N, V, U, ldu, HU, ldh, KAP, nvec, inner);
}

void launch_rayleigh(int n3, int n2, BatchRef HU, BatchRef S, int lds, BatchRef Y, int ldy, double *out, int nvec, int ncells,
                     int inner, cudaStream_t s) {
  KScope ks(KC_OTHER, 0.0, s);
  rayleigh_kernel<<<dim3(nvec, ncells * inner), 256, 0, s>>>(n3, n2, HU, S, lds, Y, ldy, out, nvec, inner);
}

}  // namespace bsk
