// S4: the coupling H(k) = V B(k), B = i(k+G) on N x N diagonal blocks (eq. 18), applied to
// Y = Phi^{-1} as an elementwise scaling:  K(k) = H^dagger Y H = V^2 Btilde(kappa)^T Y Btilde(kappa), kappa_g = k + G_g,
//   Btilde rows (s11,s22,s12) x columns (u1,u2):  [kx 0; 0 ky; ky kx]   (the i's cancel: (i kappa)^dagger (i kappa) = kappa^2).
// The kernel is bilinear in (kappa_L, kappa_R) so that the same code yields K(k) (DIRECT mode) and the six coefficient
// matrices of the polynomial K(k) = C0 + kx C1 + ky C2 + kx^2 C3 + kx ky C4 + ky^2 C5 (POLY mode).  DESIGN.md section 5.
#include "bs_internal.cuh"

namespace bsk {

namespace {
__global__ void __launch_bounds__(256) pencil_kernel(int N, double V2, BatchRef Y, int ldy, BatchRef K, int ldk,
                                                     BatchRef kvec, int nterm, int inner) {
  const int z = blockIdx.z;
  const int cell = z / inner, bi = z % inner;
  const int g = blockIdx.x * blockDim.x + threadIdx.x, h = blockIdx.y;
  if (g >= N) return;
  const cplx *__restrict__ Yg = batch_ptr(Y, cell, 0);
  cplx *Kg = batch_ptr(K, cell, bi);
  const double *__restrict__ kv = reinterpret_cast<const double *>(batch_ptr(kvec, cell, bi));
  cplx y[3][3];
#pragma unroll
  for (int b = 0; b < 3; ++b)
#pragma unroll
    for (int a = 0; a < 3; ++a) y[a][b] = Yg[(size_t)(a * N + g) + (size_t)(b * N + h) * ldy];
  cplx k11 = cmake(0, 0), k12 = k11, k21 = k11, k22 = k11;
  for (int t = 0; t < nterm; ++t) {
    const double lx = kv[((t * 2 + 0) * 2 + 0) * (size_t)N + g], ly = kv[((t * 2 + 0) * 2 + 1) * (size_t)N + g];
    const double rx = kv[((t * 2 + 1) * 2 + 0) * (size_t)N + h], ry = kv[((t * 2 + 1) * 2 + 1) * (size_t)N + h];
    const double xx = lx * rx, xy = lx * ry, yx = ly * rx, yy = ly * ry;
    // K_jl[g,h] = sum_ab BtL[a][j] Y_ab BtR[b][l]
    k11.x += xx * y[0][0].x + xy * y[0][2].x + yx * y[2][0].x + yy * y[2][2].x;
    k11.y += xx * y[0][0].y + xy * y[0][2].y + yx * y[2][0].y + yy * y[2][2].y;
    k12.x += xy * y[0][1].x + xx * y[0][2].x + yy * y[2][1].x + yx * y[2][2].x;
    k12.y += xy * y[0][1].y + xx * y[0][2].y + yy * y[2][1].y + yx * y[2][2].y;
    k21.x += yx * y[1][0].x + yy * y[1][2].x + xx * y[2][0].x + xy * y[2][2].x;
    k21.y += yx * y[1][0].y + yy * y[1][2].y + xx * y[2][0].y + xy * y[2][2].y;
    k22.x += yy * y[1][1].x + yx * y[1][2].x + xy * y[2][1].x + xx * y[2][2].x;
    k22.y += yy * y[1][1].y + yx * y[1][2].y + xy * y[2][1].y + xx * y[2][2].y;
  }
  Kg[(size_t)g + (size_t)h * ldk] = cscale(k11, V2);
  Kg[(size_t)g + (size_t)(N + h) * ldk] = cscale(k12, V2);
  Kg[(size_t)(N + g) + (size_t)h * ldk] = cscale(k21, V2);
  Kg[(size_t)(N + g) + (size_t)(N + h) * ldk] = cscale(k22, V2);
}

// A(k) = sum_i c_i(k) Coef_i on the lower triangle; one thread per entry, loops over the k-points so that the six
// coefficient entries are read once and nk results are written (HBM-write-bound).
__global__ void __launch_bounds__(256) combine_kernel(int n, BatchRef Coef, long long cstride, BatchRef Ak, int ld,
                                                      const double *__restrict__ coefk, int nk) {
  const int cell = blockIdx.z;
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n || r < c) return;
  const cplx *__restrict__ Cg = batch_ptr(Coef, cell, 0);
  const size_t e = (size_t)r + (size_t)c * ld;
  cplx v[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) v[i] = Cg[e + (size_t)i * cstride];
  for (int k = 0; k < nk; ++k) {
    const double *ck = coefk + ((size_t)cell * nk + k) * 6;
    double re = 0.0, im = 0.0;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      re = fma(ck[i], v[i].x, re);
      im = fma(ck[i], v[i].y, im);
    }
    batch_ptr(Ak, cell, k)[e] = cmake(re, im);
  }
}
}  // namespace

void launch_pencil(int N, double V2, BatchRef Y, int ldy, BatchRef K, int ldk, BatchRef kvec, int nterm, int ncells,
                   int inner, cudaStream_t s) {
  const int bs = N >= 256 ? 256 : ((N + 31) / 32) * 32;
  dim3 grid((N + bs - 1) / bs, N, ncells * inner);
  KScope ks(KC_PENCIL, 16.0 * (9.0 + 4.0) * N * N * ncells * inner, s);  // 9 blocks of Y read, 4 of K written
  pencil_kernel<<<grid, bs, 0, s>>>(N, V2, Y, ldy, K, ldk, kvec, nterm, inner);
}

void launch_combine(int n, BatchRef Coef, long long coef_mat_stride, BatchRef Ak, int ld, const double *coefk, int nk,
                    int ncells, cudaStream_t s) {
  const int bs = n >= 256 ? 256 : ((n + 31) / 32) * 32;
  dim3 grid((n + bs - 1) / bs, n, ncells);
  KScope ks(KC_COMBINE, 8.0 * n * (n + 1.0) * (6.0 + nk) * ncells, s);  // lower triangles: 6 read, nk written
  combine_kernel<<<grid, bs, 0, s>>>(n, Coef, coef_mat_stride, Ak, ld, coefk, nk);
}

}  // namespace bsk
