// S6, two-stage: (1) dense Hermitian -> Hermitian band of width b by blocked Householder QR panels whose two-sided
// trailing updates are DMMA GEMMs (this file's stage-1 driver), (2) band -> real symmetric tridiagonal by Householder
// bulge chasing in shared memory (bulge.cu).  Only eigenvalues are wanted, so no reflector is kept.
// DESIGN.md section 5 (S6).
//
// Stage 1, panel p (columns c0 = p b .. c0+b-1, rows r0 = c0+b .. n-1, m = n - r0):
//   QR      : A[r0:n, c0:c0+b] = Q R,  Q = H_1 .. H_k = I - V T V^H  (k = min(b, m-1) reflectors, V unit lower trapezoidal)
//   HEMM    : Z = A22 V                       (A22 = A[r0:n, r0:n], lower triangle read; DMMA)
//   Gram    : [G | S] = V^H [V | Z]           (b x 2b; DMMA)
//   small   : T from G and tau (forward recurrence of the compact WY form); M2 = -1/2 T^H S T
//   X       : X = Z T + V M2 = [V | Z] [M2; T]   (DMMA)            =>  Q^H A22 Q = A22 - X V^H - V X^H
//   HER2K   : A22 -= [V | X] [X | V]^H on the lower tiles           (DMMA, K = 2b)
// Workspace per matrix (VW): n x 4b complex, columns [V | X | V | Z]; SM: b x 2b (Gram) + 2b x b ([M2; T]) + b (tau).
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int QT = 1024;     // threads of the panel QR kernel (32 warps: one warp per trailing column of the panel)
constexpr int NMAXQ = 2048;  // max rows of a panel (n <= 2048)
constexpr int KS = 8;         // split-K factor of the Gram product [G | S] = V^H [V | Z] (one output tile per matrix)

__device__ __forceinline__ double block_sum_q(double x, double *scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) scratch[w] = x;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += scratch[i];
  return s;
}

// Householder QR of the m x b panel block of every matrix, right-looking, one CTA per matrix.  R overwrites the upper
// triangle of the block (the part that lies inside the band); V goes to columns [0,b) and [2b,3b) of VW (rows indexed
// globally, zeros above the unit diagonal and in unused columns); tau to SM + tau_off.
__global__ void __launch_bounds__(QT) panel_qr_kernel(int n, int lda, int b, int c0, BatchRef A, BatchRef VW, BatchRef SM,
                                                      int inner) {
  __shared__ cplx vs[NMAXQ];
  __shared__ double scratch[QT / 32];
  __shared__ cplx s_tau, s_scale;
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *Ag = batch_ptr(A, cell, mi);
  cplx *V1 = batch_ptr(VW, cell, mi);
  cplx *V2 = V1 + (size_t)2 * b * n;
  double *tau_out = reinterpret_cast<double *>(batch_ptr(SM, cell, mi) + (size_t)4 * b * b);
  const int r0 = c0 + b, m = n - r0;
  const int kq = min(b, m - 1);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  for (int j = 0; j < b; ++j) {
    cplx *colj = Ag + (size_t)(c0 + j) * lda;
    const int pr = r0 + j;  // pivot row
    if (j >= kq) {          // no reflector: V column = 0, tau = 0
      for (int r = r0 + t; r < n; r += QT) {
        V1[(size_t)j * n + r] = cmake(0.0, 0.0);
        V2[(size_t)j * n + r] = cmake(0.0, 0.0);
      }
      if (t == 0) { tau_out[2 * j] = 0.0; tau_out[2 * j + 1] = 0.0; }
      continue;
    }
    double ss = 0.0;
    for (int r = pr + 1 + t; r < n; r += QT) {
      const cplx x = colj[r];
      ss += x.x * x.x + x.y * x.y;
    }
    ss = block_sum_q(ss, scratch);
    if (t == 0) {
      const cplx al = colj[pr];
      cplx tau, scale;
      double beta;
      if (ss == 0.0 && al.y == 0.0) {
        tau = cmake(0.0, 0.0); scale = cmake(0.0, 0.0); beta = al.x;
      } else {
        beta = -copysign(sqrt(al.x * al.x + al.y * al.y + ss), al.x);
        tau = cmake((beta - al.x) / beta, -al.y / beta);
        const double dr = al.x - beta, di = al.y, den = 1.0 / (dr * dr + di * di);
        scale = cmake(dr * den, -di * den);
      }
      s_tau = tau; s_scale = scale;
      tau_out[2 * j] = tau.x; tau_out[2 * j + 1] = tau.y;
      colj[pr] = cmake(beta, 0.0);
    }
    __syncthreads();
    const cplx tau = s_tau, scale = s_scale;
    for (int r = r0 + t; r < n; r += QT) {
      cplx v = cmake(0.0, 0.0);
      if (r == pr) v = cmake(1.0, 0.0);
      else if (r > pr) v = cmul(colj[r], scale);
      vs[r - r0] = v;
      V1[(size_t)j * n + r] = v;
      V2[(size_t)j * n + r] = v;
    }
    __syncthreads();
    // apply H_j^H = I - conj(tau) v v^H to the remaining columns of the panel: one warp per column
    if (tau.x != 0.0 || tau.y != 0.0) {
      for (int c = j + 1 + warp; c < b; c += QT / 32) {
        cplx *col = Ag + (size_t)(c0 + c) * lda;
        cplx dot = cmake(0.0, 0.0), dot2 = cmake(0.0, 0.0);
        int r = pr + lane;
        for (; r + 224 < n; r += 256) {  // 8 independent 16-byte loads in flight per lane
          cplx x[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) x[u] = col[r + 32 * u];
#pragma unroll
          for (int u = 0; u < 8; u += 2) {
            cfmac(dot, vs[r + 32 * u - r0], x[u]);
            cfmac(dot2, vs[r + 32 * (u + 1) - r0], x[u + 1]);
          }
        }
        for (; r < n; r += 32) cfmac(dot, vs[r - r0], col[r]);
        dot = cadd(dot, dot2);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
          dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
        }
        const cplx f = cmul(cconj(tau), dot);
        r = pr + lane;
        for (; r + 224 < n; r += 256) {
          cplx x[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) x[u] = col[r + 32 * u];
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            cfms(x[u], vs[r + 32 * u - r0], f);
            col[r + 32 * u] = x[u];
          }
        }
        for (; r < n; r += 32) {
          cplx x = col[r];
          cfms(x, vs[r - r0], f);
          col[r] = x;
        }
      }
    }
    __syncthreads();
  }
}

// T (compact WY, forward columnwise: T[j][j] = tau_j, T[0:j, j] = -tau_j T[0:j,0:j] G[0:j, j]) and
// M2 = -1/2 T^H S T.  SM per matrix: [G | S] (b x 2b, ld b) at 0; [M2; T] (2b x b, ld 2b) at 2 b^2; tau at 4 b^2.
__global__ void __launch_bounds__(256) wy_small_kernel(int b, BatchRef SM, int inner) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *T = reinterpret_cast<cplx *>(smem_raw);  // b x b, T[i + j*b]
  cplx *S = T + b * b;                           // b x b
  cplx *U = S + b * b;                           // b x b scratch
  cplx *G = U + b * b;                           // b x b
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *sm = batch_ptr(SM, cell, mi);
  const cplx *part = sm + (size_t)4 * b * b + 64;  // KS partial products [G | S], each b x 2b
  const double *tau = reinterpret_cast<const double *>(sm + (size_t)4 * b * b);
  cplx *out = sm + (size_t)2 * b * b;
  const int t = threadIdx.x;
  for (int i = t; i < b * b; i += blockDim.x) {
    T[i] = cmake(0.0, 0.0);
    cplx gs = cmake(0.0, 0.0), ss = cmake(0.0, 0.0);
    for (int k = 0; k < KS; ++k) {  // fixed order: deterministic
      gs = cadd(gs, part[(size_t)k * 2 * b * b + i]);
      ss = cadd(ss, part[(size_t)k * 2 * b * b + b * b + i]);
    }
    G[i] = gs;
    S[i] = ss;
  }
  __syncthreads();
  for (int j = 0; j < b; ++j) {
    const cplx tj = cmake(tau[2 * j], tau[2 * j + 1]);
    if (t < j) {
      cplx acc = cmake(0.0, 0.0);
      for (int l = t; l < j; ++l) cfma(acc, T[t + l * b], G[l + j * b]);
      T[t + j * b] = cmul(cmake(-tj.x, -tj.y), acc);
    } else if (t == j) {
      T[j + j * b] = tj;
    }
    __syncthreads();
  }
  // U = S T
  for (int i = t; i < b * b; i += blockDim.x) {
    const int r = i % b, c = i / b;
    cplx acc = cmake(0.0, 0.0);
    for (int l = 0; l <= c; ++l) cfma(acc, S[r + l * b], T[l + c * b]);
    U[i] = acc;
  }
  __syncthreads();
  // M2 = -1/2 T^H U ; out = [M2; T]
  for (int i = t; i < b * b; i += blockDim.x) {
    const int r = i % b, c = i / b;
    cplx acc = cmake(0.0, 0.0);
    for (int l = 0; l <= r; ++l) cfmac(acc, T[l + r * b], U[l + c * b]);
    out[(size_t)c * 2 * b + r] = cscale(acc, -0.5);
    out[(size_t)c * 2 * b + b + r] = T[i];
  }
}

// Band extraction: AB[d + c*ldab] = A[c+d, c] for 0 <= d <= b (zero beyond the matrix and for b < d < ldab).
__global__ void __launch_bounds__(256) band_extract_kernel(int n, int lda, int b, int ldab, BatchRef A, BatchRef AB,
                                                           int inner) {
  const int z = blockIdx.z, cell = z / inner, mi = z % inner;
  const cplx *Ag = batch_ptr(A, cell, mi);
  cplx *ab = batch_ptr(AB, cell, mi);
  const int c = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (c >= n) return;
  for (int d = threadIdx.x & 31; d < ldab; d += 32) {
    cplx v = cmake(0.0, 0.0);
    if (d <= b && c + d < n) v = Ag[(size_t)(c + d) + (size_t)c * lda];
    if (d == 0) v.y = 0.0;
    ab[(size_t)c * ldab + d] = v;
  }
}
}  // namespace

size_t band_vw_elems(int n, int b) { return (size_t)4 * b * n; }
size_t band_sm_elems(int b) { return (size_t)4 * b * b + 64 + (size_t)KS * 2 * b * b; }
size_t band_ab_elems(int n, int b) { return (size_t)n * 2 * b; }

// Stage 1 for every matrix of the batch in lock step; on exit AB holds the band (ldab = 2b, bulge space zeroed).
int launch_sy2sb(int n, int lda, int b, BatchRef A, BatchRef VW, BatchRef SM, BatchRef AB, int ncells, int inner,
                 cudaStream_t s) {
  int launches = 0;
  const int nmat = ncells * inner;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(wy_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * 32 * 32 * (int)sizeof(cplx));
    attr_done = true;
  }
  for (int c0 = 0; c0 + b < n - 1; c0 += b) {
    const int r0 = c0 + b, m = n - r0;  // m >= 2
    {
      KScope ks(KC_PANEL, 0.0, s);
      panel_qr_kernel<<<nmat, QT, 0, s>>>(n, lda, b, c0, A, VW, SM, inner);
      ++launches;
    }
    GemmDesc g{};
    g.ncells = ncells; g.inner = inner; g.kclass = KC_GEMM_TRIDIAG;
    // Z = A22 V
    g.kclass = KC_GEMM_HEMM;
    g.M = m; g.N = b; g.K = m; g.opA = 0; g.opB = 0; g.flags = BS_GEMM_A_HERM_LOWER;
    g.A = A; g.A.off += (long long)r0 * (lda + 1); g.lda = lda;
    g.B = VW; g.B.off += r0; g.ldb = n;
    g.C = VW; g.C.off += (long long)3 * b * n + r0; g.ldc = n;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    launch_zgemm(g, s); ++launches;
    // [G | S] = V^H [V | Z]
    g.kclass = KC_GEMM_WY;
    g.M = b; g.N = 2 * b; g.K = m; g.opA = 1; g.opB = 0; g.flags = 0;
    g.A = VW; g.A.off += r0; g.lda = n;
    g.B = VW; g.B.off += (long long)2 * b * n + r0; g.ldb = n;
    g.C = SM; g.C.off += (long long)4 * b * b + 64; g.ldc = b;
    g.ksplit = KS; g.split_stride = (long long)2 * b * b;
    launch_zgemm(g, s); ++launches;
    g.ksplit = 0; g.split_stride = 0;
    {
      KScope ks(KC_PANEL, 0.0, s);
      wy_small_kernel<<<nmat, 256, 4 * b * b * sizeof(cplx), s>>>(b, SM, inner);
      ++launches;
    }
    // X = [V | Z] [M2; T]
    g.M = m; g.N = b; g.K = 2 * b; g.opA = 0; g.opB = 0; g.flags = 0;
    g.A = VW; g.A.off += (long long)2 * b * n + r0; g.lda = n;
    g.B = SM; g.B.off += (long long)2 * b * b; g.ldb = 2 * b;
    g.C = VW; g.C.off += (long long)b * n + r0; g.ldc = n;
    launch_zgemm(g, s); ++launches;
    // A22 -= [V | X] [X | V]^H  (lower tiles)
    g.kclass = KC_GEMM_TRIDIAG;
    g.M = m; g.N = m; g.K = 2 * b; g.opA = 0; g.opB = 1; g.flags = BS_GEMM_LOWER_ONLY;
    g.A = VW; g.A.off += r0; g.lda = n;
    g.B = VW; g.B.off += (long long)b * n + r0; g.ldb = n;
    g.C = A; g.C.off += (long long)r0 * (lda + 1); g.ldc = lda;
    g.alpha = cmake(-1.0, 0.0); g.beta = cmake(1.0, 0.0);
    launch_zgemm(g, s); ++launches;
  }
  {
    KScope ks(KC_OTHER, 0.0, s);
    band_extract_kernel<<<dim3((n + 7) / 8, 1, nmat), 256, 0, s>>>(n, lda, b, 2 * b, A, AB, inner);
    ++launches;
  }
  return launches;
}

}  // namespace bsk
