// S3: blocked lower Cholesky (right-looking, 64-wide panels) and triangular inverse by recursive doubling; both push
// their flops through the DMMA zgemm.  Implied by PAPER.md:101 (eq. 11: Phi^{-1}); DESIGN.md section 5 (factor).
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int NB = 64;
constexpr int LDP = NB + 1;

__host__ BatchRef shifted(BatchRef r, long long delta) {
  r.off += delta;
  return r;
}

// Factor the diagonal block [j0, j0+nbk) of every matrix in shared memory and also produce its inverse.
//   A    : n x n (lda), lower.  On exit the block holds L11 (strict upper part of the block zeroed).
//   dinv : block jb of the per-matrix array of 64x64 inverses (column-major, ld 64, zeros above the diagonal).
__global__ void __launch_bounds__(256) potrf_diag_kernel(int n, int lda, int j0, BatchRef A, BatchRef dinv, int *info) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx(*S)[LDP] = reinterpret_cast<cplx(*)[LDP]>(smem_raw);                      // S[col][row]
  cplx(*X)[LDP] = reinterpret_cast<cplx(*)[LDP]>(smem_raw + sizeof(cplx) * NB * LDP);
  const int cell = blockIdx.z;
  cplx *Ag = batch_ptr(A, cell, 0) + (size_t)j0 + (size_t)j0 * lda;
  cplx *Dg = batch_ptr(dinv, cell, 0) + (size_t)(j0 / NB) * NB * NB;
  const int nbk = min(NB, n - j0);
  const int t = threadIdx.x;

  for (int i = t; i < NB * NB; i += blockDim.x) {
    const int r = i % NB, c = i / NB;
    cplx v = cmake(0.0, 0.0);
    if (r < nbk && c < nbk && r >= c) v = Ag[(size_t)r + (size_t)c * lda];
    S[c][r] = v;
    X[c][r] = cmake(0.0, 0.0);
  }
  __syncthreads();
  // thread (r, g): row r = t & 63, column group g = t >> 6 (columns c+1+g, c+5+g, ...)
  const int r = t & (NB - 1), g = t >> 6;
  for (int c = 0; c < nbk; ++c) {
    if (t == 0) {
      double piv = S[c][c].x;
      if (!(piv > 0.0)) {
        if (info[cell] == 0) info[cell] = j0 + c + 1;
        piv = 1.0;
      }
      S[c][c] = cmake(sqrt(piv), 0.0);
    }
    __syncthreads();
    const double dinvc = 1.0 / S[c][c].x;
    if (g == 0 && r > c && r < nbk) S[c][r] = cscale(S[c][r], dinvc);
    __syncthreads();
    // trailing update of the block: S[cc][r] -= S[c][r] conj(S[c][cc]),  c < cc <= r
    if (r > c && r < nbk) {
      const cplx lr = S[c][r];
      for (int cc = c + 1 + g; cc <= r; cc += 4) {
        cplx v = S[cc][r];
        cfms(v, lr, cconj(S[c][cc]));
        S[cc][r] = v;
      }
    }
    __syncthreads();
  }
  // X = L^{-1} row by row: X[r][c] = -(1/L[r][r]) sum_{k=c}^{r-1} L[r][k] X[k][c]; thread (c, g) sums k = c+g, c+g+4, ...
  __shared__ cplx psum[4][NB];
  if (g == 0 && r < nbk) X[r][r] = cmake(1.0 / S[r][r].x, 0.0);
  __syncthreads();
  for (int rr = 1; rr < nbk; ++rr) {
    const int c = r;
    cplx acc = cmake(0.0, 0.0);
    if (c < rr)
      for (int k = c + g; k < rr; k += 4) cfma(acc, S[k][rr], X[c][k]);
    psum[g][c] = acc;
    __syncthreads();
    if (g == 0 && c < rr) {
      const cplx sum = cadd(cadd(psum[0][c], psum[1][c]), cadd(psum[2][c], psum[3][c]));
      X[c][rr] = cscale(sum, -1.0 / S[rr][rr].x);
    }
    __syncthreads();
  }
  for (int i = t; i < NB * NB; i += blockDim.x) {
    const int r = i % NB, c = i / NB;
    if (r < nbk && c < nbk) Ag[(size_t)r + (size_t)c * lda] = S[c][r];  // zeros above the diagonal of the block
    Dg[i] = X[c][r];
  }
}

// X := blockdiag(dinv) (zeros elsewhere), n x n, ld = lda.
__global__ void __launch_bounds__(256) trtri_init_kernel(int n, int lda, BatchRef X, BatchRef dinv) {
  const int cell = blockIdx.z;
  cplx *Xg = batch_ptr(X, cell, 0);
  const cplx *Dg = batch_ptr(dinv, cell, 0);
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n) return;
  cplx v = cmake(0.0, 0.0);
  if (r / NB == c / NB) v = Dg[(size_t)(c / NB) * NB * NB + (size_t)(c % NB) * NB + (r % NB)];
  Xg[(size_t)r + (size_t)c * lda] = v;
}

__global__ void __launch_bounds__(256) copy_matrix_kernel(int rows, int cols, BatchRef src, int lds, BatchRef dst, int ldd,
                                                          int inner) {
  const int cell = blockIdx.z / inner, bi = blockIdx.z % inner;
  const cplx *S = batch_ptr(src, cell, bi);
  cplx *D = batch_ptr(dst, cell, bi);
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r < rows) D[(size_t)r + (size_t)c * ldd] = S[(size_t)r + (size_t)c * lds];
}

// A[c][r] := conj(A[r][c]) for r > c (mirror the lower triangle), 32x32 tiles through shared memory.
__global__ void __launch_bounds__(256) fill_upper_kernel(int n, BatchRef A, int lda, int inner) {
  __shared__ cplx tile[32][33];
  const int bi = blockIdx.x, bj = blockIdx.y;  // tile (rows bi, cols bj) of the LOWER triangle, bi >= bj
  if (bi < bj) return;
  const int cell = blockIdx.z / inner, ii = blockIdx.z % inner;
  cplx *Ag = batch_ptr(A, cell, ii);
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int cc = ty; cc < 32; cc += 8) {
    const int r = bi * 32 + tx, c = bj * 32 + cc;
    if (r < n && c < n) tile[cc][tx] = Ag[(size_t)r + (size_t)c * lda];
  }
  __syncthreads();
  for (int rr = ty; rr < 32; rr += 8) {
    // destination (row = bj*32 + tx, col = bi*32 + rr) <- conj(source (row = bi*32+rr, col = bj*32+tx))
    const int dr = bj * 32 + tx, dc = bi * 32 + rr;
    if (dr < n && dc < n && dc > dr) Ag[(size_t)dr + (size_t)dc * lda] = cconj(tile[tx][rr]);
  }
}
}  // namespace

void launch_copy_matrix(int rows, int cols, BatchRef src, int lds, BatchRef dst, int ldd, int ncells, int inner,
                        cudaStream_t s) {
  dim3 grid((rows + 255) / 256, cols, ncells * inner);
  copy_matrix_kernel<<<grid, 256, 0, s>>>(rows, cols, src, lds, dst, ldd, inner);
}

void launch_hermitian_fill_upper(int n, BatchRef A, int lda, int ncells, int inner, cudaStream_t s) {
  const int nt = (n + 31) / 32;
  dim3 grid(nt, nt, ncells * inner);
  fill_upper_kernel<<<grid, 256, 0, s>>>(n, A, lda, inner);
}

int potrf_trtri(int n, int lda, BatchRef A, BatchRef X, BatchRef tmp, BatchRef dinv, int *info, long long, int ncells,
                int inner_unused, cudaStream_t s) {
  (void)inner_unused;
  int launches = 0;
  const size_t diag_smem = sizeof(cplx) * NB * LDP * 2;
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(potrf_diag_kernel, (int)diag_smem, attr_mask);
  // ---- Cholesky, right-looking
  for (int j0 = 0; j0 < n; j0 += NB) {
    const int nbk = n - j0 < NB ? n - j0 : NB;
    { KScope ks(KC_POTRF_DIAG, 0.0, s);
      potrf_diag_kernel<<<dim3(1, 1, ncells), 256, diag_smem, s>>>(n, lda, j0, A, dinv, info); }
    ++launches;
    const int r = n - j0 - nbk;
    if (r <= 0) break;
    GemmDesc g{};
    g.ncells = ncells; g.inner = 1; g.kclass = KC_GEMM_FACTOR;
    // A21 <- A21 * inv(L11)^dagger
    g.M = r; g.N = nbk; g.K = nbk; g.opA = 0; g.opB = 1;
    g.A = shifted(A, (long long)(j0 + nbk) + (long long)j0 * lda); g.lda = lda;
    g.B = shifted(dinv, (long long)(j0 / NB) * NB * NB); g.ldb = NB;
    g.C = g.A; g.ldc = lda;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0); g.flags = 0;
    launch_zgemm(g, s);
    ++launches;
    // A22 <- A22 - A21 A21^dagger (lower tiles)
    g.M = r; g.N = r; g.K = nbk; g.opA = 0; g.opB = 1;
    g.B = g.A; g.ldb = lda;
    g.C = shifted(A, (long long)(j0 + nbk) * (lda + 1)); g.ldc = lda;
    g.alpha = cmake(-1.0, 0.0); g.beta = cmake(1.0, 0.0); g.flags = BS_GEMM_LOWER_ONLY;
    launch_zgemm(g, s);
    ++launches;
  }
  // ---- X = L^{-1} by recursive doubling: [L11 0; L21 L22]^{-1} = [X11 0; -X22 L21 X11, X22]
  trtri_init_kernel<<<dim3((n + 255) / 256, n, ncells), 256, 0, s>>>(n, lda, X, dinv);
  ++launches;
  for (int sz = NB; sz < n; sz *= 2) {
    const int npair_full = n / (2 * sz);               // pairs whose second block is complete
    const int rem = n - npair_full * 2 * sz;            // what is left after the full pairs
    for (int pass = 0; pass < 2; ++pass) {
      int r0, s2, cnt;
      if (pass == 0) { r0 = 0; s2 = sz; cnt = npair_full; }
      else { r0 = npair_full * 2 * sz; s2 = rem - sz; cnt = 1; }  // one partial pair if rem > sz
      if (cnt <= 0 || s2 <= 0) continue;
      const long long pstride = (long long)2 * sz * (lda + 1);
      GemmDesc g{};
      g.ncells = ncells; g.inner = cnt; g.kclass = KC_GEMM_FACTOR;
      // T = L21 X11   (X11 lower: k >= n)
      g.M = s2; g.N = sz; g.K = sz; g.opA = 0; g.opB = 0;
      g.A = shifted(A, (long long)(r0 + sz) + (long long)r0 * lda); g.A.stride = pstride; g.lda = lda;
      g.B = shifted(X, (long long)r0 * (lda + 1)); g.B.stride = pstride; g.ldb = lda;
      g.C = shifted(tmp, (long long)(r0 + sz) + (long long)r0 * lda); g.C.stride = pstride; g.ldc = lda;
      g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0); g.flags = BS_GEMM_KLO_COL;
      launch_zgemm(g, s);
      ++launches;
      // X21 = -X22 T  (X22 lower: k <= m)
      g.M = s2; g.N = sz; g.K = s2;
      g.A = shifted(X, (long long)(r0 + sz) * (lda + 1)); g.A.stride = pstride; g.lda = lda;
      g.B = g.C; g.ldb = lda;
      g.C = shifted(X, (long long)(r0 + sz) + (long long)r0 * lda); g.C.stride = pstride; g.ldc = lda;
      g.alpha = cmake(-1.0, 0.0); g.flags = BS_GEMM_KHI_ROW;
      launch_zgemm(g, s);
      ++launches;
    }
  }
  return launches;
}

}  // namespace bsk
