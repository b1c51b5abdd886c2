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
constexpr int KS = 8;         // split-K factor of the Gram product [G | S] = V^H [V | Z] (one output tile per matrix)

// Householder QR of the m x b panel block of every matrix, one CTA per matrix.  The panel is processed in sub-panels
// of SW = 4 columns held in shared memory: a sub-panel is factored there (no global round trips between its columns), its
// four reflectors are then applied to the remaining panel columns as one compact-WY update (two passes over each column
// instead of eight; one warp per column).  R overwrites the upper triangle of the block (the part that lies inside the
// band); V goes to columns [0,b) and [2b,3b) of VW (rows indexed globally, zeros above the unit diagonal and in unused
// columns); tau to SM + 4 b^2.
constexpr int SW = 4;  // sub-panel width

template <int K, int NTHR>
__device__ __forceinline__ void block_reduce(double (&v)[K], double *red, double *res) {
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
  if (warp == 0) {
#pragma unroll
    for (int k = 0; k < K; ++k) {
      double x = lane < NTHR / 32 ? red[lane * K + k] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
      if (lane == 0) res[k] = x;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) v[k] = res[k];
  // no third barrier: the next reduction writes `res` only after its own first barrier, which every thread reaches
  // after these reads; its `red` writes come after this reduction's second barrier
}

// MINB: resident CTAs per SM the register allocation must allow (256-thread variant): 2 when a few matrices each wait on
// their own latency chain (128 registers), 4 when the batch is large and the SM is shared (64 registers, throughput).
template <int NTHR, int MINB = 1>
__global__ void __launch_bounds__(NTHR, MINB) panel_qr_kernel(int n, int lda, int b, int c0, BatchRef A, BatchRef VW, BatchRef SM,
                                                        int inner) {
  extern __shared__ __align__(16) unsigned char qr_smem[];
  const int r0 = c0 + b, m = n - r0;
  cplx *sp = reinterpret_cast<cplx *>(qr_smem);                 // [SW][m]
  double *red = reinterpret_cast<double *>(sp + (size_t)SW * m);  // [NTHR/32][32]
  double *res = red + (NTHR / 32) * 32;                           // [32]
  cplx *scal = reinterpret_cast<cplx *>(res + 32);                // tau, scale, then T (SW x SW)
  cplx *Tm = scal + 2;
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *Ag = batch_ptr(A, cell, mi);
  cplx *V1 = batch_ptr(VW, cell, mi);
  cplx *V2 = V1 + (size_t)2 * b * n;
  double *tau_out = reinterpret_cast<double *>(batch_ptr(SM, cell, mi) + (size_t)4 * b * b);
  const int kq = min(b, m - 1);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

  for (int js = 0; js < b; js += SW) {
    // 1. sub-panel -> shared memory
    for (int q = t; q < SW * m; q += NTHR) {
      const int jj = q / m, i = q % m;
      sp[q] = Ag[(size_t)(r0 + i) + (size_t)(c0 + js + jj) * lda];
    }
    __syncthreads();
    cplx taus[SW];
    double nxt = -1.0;  // partial sum of |x|^2 below the pivot of the next column, gathered while it is updated
    // 2. factor it
#pragma unroll
    for (int jj = 0; jj < SW; ++jj) {
      const int j = js + jj;  // local pivot index = j
      cplx *cj = sp + (size_t)jj * m;
      cplx *gj = Ag + (size_t)(c0 + j) * lda + r0;
      if (j >= kq) {  // nothing below the pivot: the whole column is R; no reflector
        for (int i = t; i < m; i += NTHR) { gj[i] = cj[i]; }
        __syncthreads();
        for (int i = t; i < m; i += NTHR) cj[i] = cmake(0.0, 0.0);
        if (t == 0) { tau_out[2 * j] = 0.0; tau_out[2 * j + 1] = 0.0; }
        taus[jj] = cmake(0.0, 0.0);
        __syncthreads();
        continue;
      }
      double nv[1] = {0.0};
      if (nxt >= 0.0) nv[0] = nxt;
      else for (int i = j + 1 + t; i < m; i += NTHR) { const cplx x = cj[i]; nv[0] += x.x * x.x + x.y * x.y; }
      nxt = -1.0;
      block_reduce<1, NTHR>(nv, red, res);
      if (t == 0) {
        const cplx al = cj[j];
        const double ss = nv[0];
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
        scal[0] = tau; scal[1] = scale;
        tau_out[2 * j] = tau.x; tau_out[2 * j + 1] = tau.y;
        gj[j] = cmake(beta, 0.0);  // R diagonal
      }
      __syncthreads();
      const cplx tau = scal[0], scale = scal[1];
      taus[jj] = tau;
      // R entries above the pivot go home; the column becomes v (zeros above, 1 at the pivot)
      double dv[2 * (SW - 1)];
#pragma unroll
      for (int k = 0; k < 2 * (SW - 1); ++k) dv[k] = 0.0;
      for (int i = t; i < m; i += NTHR) {
        cplx v;
        if (i < j) { gj[i] = cj[i]; v = cmake(0.0, 0.0); }
        else if (i == j) v = cmake(1.0, 0.0);
        else v = cmul(cj[i], scale);
        cj[i] = v;
        if (i >= j) {
#pragma unroll
          for (int kk = jj + 1; kk < SW; ++kk) {
            const cplx x = sp[(size_t)kk * m + i];
            dv[2 * (kk - 1)] += v.x * x.x + v.y * x.y;      // conj(v) x
            dv[2 * (kk - 1) + 1] += v.x * x.y - v.y * x.x;
          }
        }
      }
      if (jj + 1 < SW) {
        block_reduce<2 * (SW - 1), NTHR>(dv, red, res);
        nxt = 0.0;
        for (int i = j + t; i < m; i += NTHR) {
          const cplx v = cj[i];
#pragma unroll
          for (int kk = jj + 1; kk < SW; ++kk) {
            const cplx f = cmul(cconj(tau), cmake(dv[2 * (kk - 1)], dv[2 * (kk - 1) + 1]));
            cplx x = sp[(size_t)kk * m + i];
            cfms(x, v, f);
            sp[(size_t)kk * m + i] = x;
            if (kk == jj + 1 && i > j + 1) nxt += x.x * x.x + x.y * x.y;
          }
        }
        if (j + 1 >= kq) nxt = -1.0;  // the next column has no reflector
      }
      __syncthreads();
    }
    // 3. Gram entries v_a^H v_b (a < b) -> T of the sub-panel (forward columnwise compact WY)
    {
      double gv[12];
#pragma unroll
      for (int k = 0; k < 12; ++k) gv[k] = 0.0;
      for (int i = js + t; i < m; i += NTHR) {
        cplx v[SW];
#pragma unroll
        for (int jj = 0; jj < SW; ++jj) v[jj] = sp[(size_t)jj * m + i];
        int e = 0;
#pragma unroll
        for (int a = 0; a < SW; ++a)
#pragma unroll
          for (int c = a + 1; c < SW; ++c) {
            gv[2 * e] += v[a].x * v[c].x + v[a].y * v[c].y;
            gv[2 * e + 1] += v[a].x * v[c].y - v[a].y * v[c].x;
            ++e;
          }
      }
      block_reduce<12, NTHR>(gv, red, res);
      if (t == 0) {
        cplx Gm[SW][SW];
        int e = 0;
        for (int a = 0; a < SW; ++a)
          for (int c = a + 1; c < SW; ++c) { Gm[a][c] = cmake(gv[2 * e], gv[2 * e + 1]); ++e; }
        cplx Tl[SW][SW];
        for (int a = 0; a < SW; ++a)
          for (int c = 0; c < SW; ++c) Tl[a][c] = cmake(0.0, 0.0);
        for (int c = 0; c < SW; ++c) {
          Tl[c][c] = taus[c];
          for (int a = 0; a < c; ++a) {
            cplx acc = cmake(0.0, 0.0);
            for (int l2 = a; l2 < c; ++l2) cfma(acc, Tl[a][l2], Gm[l2][c]);
            Tl[a][c] = cmul(cmake(-taus[c].x, -taus[c].y), acc);
          }
        }
        for (int a = 0; a < SW; ++a)
          for (int c = 0; c < SW; ++c) Tm[a * SW + c] = Tl[a][c];
      }
    }
    // 4. V columns out
    for (int q = t; q < SW * m; q += NTHR) {
      const int jj = q / m, i = q % m;
      const cplx v = sp[q];
      V1[(size_t)(js + jj) * n + r0 + i] = v;
      V2[(size_t)(js + jj) * n + r0 + i] = v;
    }
    __syncthreads();  // Tm visible
    // 5. remaining panel columns: x <- x - V T^H (V^H x), one warp per column, rows >= js
    cplx Tr[SW][SW];
#pragma unroll
    for (int a = 0; a < SW; ++a)
#pragma unroll
      for (int c = 0; c < SW; ++c) Tr[a][c] = Tm[a * SW + c];
    for (int c = js + SW + warp; c < b; c += NTHR / 32) {
      cplx *col = Ag + (size_t)(c0 + c) * lda + r0;
      cplx d[SW];
#pragma unroll
      for (int k = 0; k < SW; ++k) d[k] = cmake(0.0, 0.0);
      int i = js + lane;
      for (; i + 96 < m; i += 128) {  // 4 independent loads in flight per lane
        cplx x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) x[u] = col[i + 32 * u];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
          for (int k = 0; k < SW; ++k) cfmac(d[k], sp[(size_t)k * m + i + 32 * u], x[u]);
      }
      for (; i < m; i += 32) {
        const cplx x = col[i];
#pragma unroll
        for (int k = 0; k < SW; ++k) cfmac(d[k], sp[(size_t)k * m + i], x);
      }
#pragma unroll
      for (int k = 0; k < SW; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          d[k].x += __shfl_xor_sync(0xffffffffu, d[k].x, o);
          d[k].y += __shfl_xor_sync(0xffffffffu, d[k].y, o);
        }
      }
      cplx gk[SW];  // g = T^H d
#pragma unroll
      for (int k = 0; k < SW; ++k) {
        gk[k] = cmake(0.0, 0.0);
#pragma unroll
        for (int l2 = 0; l2 <= k; ++l2) cfmac(gk[k], Tr[l2][k], d[l2]);
      }
      i = js + lane;
      for (; i + 96 < m; i += 128) {
        cplx x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) x[u] = col[i + 32 * u];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
          for (int k = 0; k < SW; ++k) cfms(x[u], sp[(size_t)k * m + i + 32 * u], gk[k]);
          col[i + 32 * u] = x[u];
        }
      }
      for (; i < m; i += 32) {
        cplx x = col[i];
#pragma unroll
        for (int k = 0; k < SW; ++k) cfms(x, sp[(size_t)k * m + i], gk[k]);
        col[i] = x;
      }
    }
    __syncthreads();
  }
}

// T (compact WY, forward columnwise: Q = H_1 .. H_b = I - V T V^H) and M2 = -1/2 T^H S T.
// T^-1 = diag(1 / tau) + triu(G, 1) with G = V^H V, so T solves  (I + diag(tau) triu(G, 1)) T = diag(tau):  all b columns
// at once by column-oriented back substitution, one barrier per row l = b-1 .. 0 and O(1) work per thread and step
// (R: running right-hand sides; row l of T is final at step l: T[l, j] = tau_l R[l, j], then R[i, j] -= G[i, l] T[l, j]
// for i < l).  tau_l = 0 (H_l = I) gives a zero row and column, as the forward recurrence does.
// SM per matrix: [G | S] (b x 2b, ld b) at 0; [M2; T] (2b x b, ld 2b) at 2 b^2; tau at 4 b^2.
__global__ void __launch_bounds__(1024) wy_small_kernel(int b, BatchRef SM, int inner) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *T = reinterpret_cast<cplx *>(smem_raw);  // b x b, T[i + j*b]
  cplx *S = T + b * b;                           // b x b
  cplx *U = S + b * b;                           // b x b scratch: R during the substitution, then S T
  cplx *G = U + b * b;                           // b x b
  cplx *taus = G + b * b;                        // b
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *sm = batch_ptr(SM, cell, mi);
  const cplx *part = sm + (size_t)4 * b * b + 64;  // KS partial products [G | S], each b x 2b
  cplx *out = sm + (size_t)2 * b * b;
  const int t = threadIdx.x;
  if (t < b) taus[t] = sm[(size_t)4 * b * b + t];
  for (int i = t; i < b * b; i += blockDim.x) {
    cplx gs = cmake(0.0, 0.0), ss = cmake(0.0, 0.0);
    for (int k = 0; k < KS; ++k) {  // fixed order: deterministic
      gs = cadd(gs, part[(size_t)k * 2 * b * b + i]);
      ss = cadd(ss, part[(size_t)k * 2 * b * b + b * b + i]);
    }
    G[i] = gs;
    S[i] = ss;
    T[i] = cmake(0.0, 0.0);
    U[i] = (i % b == i / b) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
  }
  __syncthreads();
  for (int l = b - 1; l >= 0; --l) {
    const cplx tl = taus[l];
    for (int e = t; e < b * b; e += blockDim.x) {
      const int i = e % b, j = e / b;
      if (j < l || i > l) continue;
      const cplx x = cmul(tl, U[l + j * b]);  // T[l, j]
      if (i == l) T[e] = x;
      else { cplx r = U[e]; cfms(r, G[i + l * b], x); U[e] = r; }
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
                 cudaStream_t s, const BatchRef *keepV, const BatchRef *keepT) {
  int launches = 0;
  const int nmat = ncells * inner;
  static unsigned long long m1 = 0, m2 = 0, m3 = 0, m4 = 0;
  ensure_dyn_smem(panel_qr_kernel<1024>, 140 * 1024, m1);
  ensure_dyn_smem(panel_qr_kernel<256, 2>, 48 * 1024, m2);
  ensure_dyn_smem(panel_qr_kernel<256, 4>, 48 * 1024, m3);
  ensure_dyn_smem(wy_small_kernel, (4 * 32 * 32 + 32) * (int)sizeof(cplx), m4);
  for (int c0 = 0; c0 + b < n - 1; c0 += b) {
    const int r0 = c0 + b, m = n - r0;  // m >= 2
    {
      KScope ks(KC_PANEL, 0.0, s);
      if (m > 640) {
        const size_t smem = (size_t)SW * m * sizeof(cplx) + (32 * 32 + 32) * sizeof(double) + (2 + SW * SW) * sizeof(cplx);
        panel_qr_kernel<1024><<<nmat, 1024, smem, s>>>(n, lda, b, c0, A, VW, SM, inner);
      } else {
        const size_t smem = (size_t)SW * m * sizeof(cplx) + (8 * 32 + 32) * sizeof(double) + (2 + SW * SW) * sizeof(cplx);
        if (nmat > 592) panel_qr_kernel<256, 4><<<nmat, 256, smem, s>>>(n, lda, b, c0, A, VW, SM, inner);
        else panel_qr_kernel<256, 2><<<nmat, 256, smem, s>>>(n, lda, b, c0, A, VW, SM, inner);
      }
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
      KScope ks(KC_OTHER, 0.0, s);
      // few matrices: one thread per entry (latency); many: smaller CTAs, several per SM (throughput)
      wy_small_kernel<<<nmat, nmat > 592 ? 256 : b * b, (4 * b * b + b) * sizeof(cplx), s>>>(b, SM, inner);
      ++launches;
    }
    if (keepV) {  // mode shapes: V and T of this panel are needed again for the back-transformation
      BatchRef src = VW, dst = *keepV;
      src.off += r0;
      dst.off += (long long)c0 * n + r0;
      launch_copy_matrix(m, b, src, n, dst, n, ncells, inner, s); ++launches;
      src = SM; src.off += (long long)2 * b * b + b;   // T inside [M2; T] (ld 2b)
      dst = *keepT; dst.off += (long long)(c0 / b) * b * b;
      launch_copy_matrix(b, b, src, 2 * b, dst, b, ncells, inner, s); ++launches;
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
