// S6: batched Householder tridiagonalisation Q^H A Q = T of Hermitian matrices (lower triangle authoritative), the
// blocked one-stage scheme (panel of nb reflectors, then one Hermitian rank-2nb update A22 -= V W^H + W V^H that runs on
// the DMMA zgemm).  Solves the pencil of PAPER.md:94-104 (eq. 10-11) after the Psi-reduction; DESIGN.md section 5 (S6).
//
// Per column j of a panel (panel index i):
//   reflect : a_j = A[j:n, j] - V[j:n,0:i] W[j,0:i]^H - W[j:n,0:i] V[j,0:i]^H ; d_j = Re a_j[0];
//             (tau, v, beta) = Householder of a_j[1:]  (v[0] = 1, H = I - tau v v^H, H^H x = beta e_1, beta real); e_j = beta
//   hemv    : y = A22 v            (A22 = A[j+1:n, j+1:n], not yet updated by this panel), tile partial sums, lower only
//   finish  : w = tau (y - V (W^H v) - W (V^H v)) ; w += (-tau/2 (w^H v)) v
// Only eigenvalues are wanted, so reflectors are not stored back into A.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int TS = 64;   // hemv tile edge
constexpr int NT = 256;  // hemv threads
constexpr int PT = 512;  // panel-step threads
constexpr int NMAX = 2048;
constexpr size_t kHemvSmem = sizeof(cplx) * (TS * (TS + 1) + 2 * TS + 2 * 4 * TS);

// ---------------------------------------------------------------- hemv partial sums
// grid (nt, nt, nmat), tile (bi, bj) = (tb0 + blockIdx.x, tb0 + blockIdx.y), bi >= bj.  P: [nblk][nblk*TS] per matrix.
__global__ void __launch_bounds__(NT) hemv_kernel(int n, int lda, int j, int tb0, int nblk, BatchRef A, BatchRef VW, int vcol,
                                                  BatchRef P, int inner) {
  const int bi = tb0 + blockIdx.x, bj = tb0 + blockIdx.y;
  if (bj > bi) return;
  extern __shared__ __align__(16) unsigned char hemv_smem[];
  cplx(*S)[TS + 1] = reinterpret_cast<cplx(*)[TS + 1]>(hemv_smem);
  cplx *vr = reinterpret_cast<cplx *>(hemv_smem) + TS * (TS + 1), *vc = vr + TS;
  cplx(*red)[4][TS] = reinterpret_cast<cplx(*)[4][TS]>(vc + TS);
  const int cell = blockIdx.z / inner, mi = blockIdx.z % inner;
  const cplx *__restrict__ Ag = batch_ptr(A, cell, mi);
  const cplx *__restrict__ v = batch_ptr(VW, cell, mi) + (size_t)vcol * n;
  cplx *Pg = batch_ptr(P, cell, mi);
  const int t = threadIdx.x, r = t & (TS - 1), q = t >> 6;
  const int npad = nblk * TS;
  if (t < TS) {
    const int row = bi * TS + t;
    vr[t] = (row < n && row > j) ? v[row] : cmake(0.0, 0.0);
  } else if (t < 2 * TS) {
    const int col = bj * TS + (t - TS);
    vc[t - TS] = (col < n && col > j) ? v[col] : cmake(0.0, 0.0);
  }
  const int row = bi * TS + r;
  cplx a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int c = q * 16 + k, col = bj * TS + c;
    const bool ok = row < n && col < n && row >= col && col > j;
    cplx x = ok ? Ag[(size_t)row + (size_t)col * lda] : cmake(0.0, 0.0);
    if (row == col) x.y = 0.0;
    a[k] = x;
    S[c][r] = x;
  }
  __syncthreads();
  cplx accr = cmake(0.0, 0.0), accc = cmake(0.0, 0.0);
#pragma unroll
  for (int k = 0; k < 16; ++k) cfma(accr, a[k], vc[q * 16 + k]);
  {
    const int c = r;  // this thread's column in the transposed pass
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int rr = q * 16 + k;
      if (bi != bj || rr != c) cfmac(accc, S[c][rr], vr[rr]);
    }
  }
  red[0][q][r] = accr;
  red[1][q][r] = accc;
  __syncthreads();
  if (t < 2 * TS) {
    const int which = t >> 6, x = t & (TS - 1);
    cplx s = cadd(cadd(red[which][0][x], red[which][1][x]), cadd(red[which][2][x], red[which][3][x]));
    if (bi == bj) {
      if (which == 0) {
        const cplx s2 = cadd(cadd(red[1][0][x], red[1][1][x]), cadd(red[1][2][x], red[1][3][x]));
        Pg[(size_t)bi * npad + bi * TS + x] = cadd(s, s2);
      }
    } else if (which == 0) {
      Pg[(size_t)bj * npad + bi * TS + x] = s;  // rows of block bi, slot bj
    } else {
      Pg[(size_t)bi * npad + bj * TS + x] = s;  // rows of block bj, slot bi
    }
  }
}

__device__ __forceinline__ double block_sum(double x, double *scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) scratch[w] = x;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += scratch[i];  // same order in every thread: deterministic
  return s;
}

// ---------------------------------------------------------------- panel step: finish w_{i-1}, then reflect column i
// One CTA per matrix.  VW per matrix: [V (n x nb) | W (n x nb) | V again (n x nb)], ld n (the copy makes [V W] and [W V]
// contiguous operands of the rank-2nb update).  scal per matrix: [0..1] = tau of the pending reflector.
__global__ void __launch_bounds__(PT) panel_step_kernel(int n, int lda, int nb, int j0, int ifin, int iref, int tb0_fin,
                                                        int nblk, BatchRef A, BatchRef VW, BatchRef P, double *d, double *e,
                                                        double *scal, int inner) {
  __shared__ cplx y[NMAX];
  __shared__ cplx t1[32], t2[32];
  __shared__ double scratch[PT / 32];
  const int z = blockIdx.x;
  const int cell = z / inner, mi = z % inner;
  const cplx *__restrict__ Ag = batch_ptr(A, cell, mi);
  cplx *V = batch_ptr(VW, cell, mi);
  cplx *W = V + (size_t)nb * n;
  cplx *V2 = W + (size_t)nb * n;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

  if (ifin >= 0) {  // ---- finish w for panel column ifin (global column j)
    const int i = ifin, j = j0 + i;
    const cplx *Pg = batch_ptr(P, cell, mi);
    const int npad = nblk * TS;
    const cplx tau = cmake(scal[2 * z], scal[2 * z + 1]);
    const cplx *v = V + (size_t)i * n;
    // t1 = W^H v, t2 = V^H v over rows > j  (one warp per dot product)
    for (int k = warp; k < 2 * i; k += PT / 32) {
      const cplx *col = (k < i) ? W + (size_t)k * n : V + (size_t)(k - i) * n;
      cplx acc = cmake(0.0, 0.0);
      for (int r = j + 1 + lane; r < n; r += 32) cfmac(acc, col[r], v[r]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
      }
      if (lane == 0) {
        if (k < i) t1[k] = acc; else t2[k - i] = acc;
      }
    }
    __syncthreads();
    double dre = 0.0, dim = 0.0;  // w^H v
    for (int r = j + 1 + t; r < n; r += PT) {
      cplx s = cmake(0.0, 0.0);
      for (int sl = tb0_fin; sl < nblk; ++sl) s = cadd(s, Pg[(size_t)sl * npad + r]);
      for (int k = 0; k < i; ++k) {
        cfms(s, V[(size_t)k * n + r], t1[k]);
        cfms(s, W[(size_t)k * n + r], t2[k]);
      }
      s = cmul(tau, s);
      y[r] = s;
      const cplx vv = v[r];
      dre += s.x * vv.x + s.y * vv.y;   // conj(w) * v
      dim += s.x * vv.y - s.y * vv.x;
    }
    dre = block_sum(dre, scratch);
    dim = block_sum(dim, scratch);
    const cplx alpha = cmul(cmake(-0.5 * tau.x, -0.5 * tau.y), cmake(dre, dim));
    for (int r = j + 1 + t; r < n; r += PT) {
      cplx s = y[r];
      cfma(s, alpha, v[r]);
      W[(size_t)i * n + r] = s;
    }
    __syncthreads();
  }
  if (iref >= 0) {  // ---- updated column j and its reflector
    const int i = iref, j = j0 + i;
    if (t < i) {
      t1[t] = cconj(W[(size_t)t * n + j]);
      t2[t] = cconj(V[(size_t)t * n + j]);
    }
    __syncthreads();
    double ss = 0.0;
    for (int r = j + t; r < n; r += PT) {
      cplx s = Ag[(size_t)r + (size_t)j * lda];
      for (int k = 0; k < i; ++k) {
        cfms(s, V[(size_t)k * n + r], t1[k]);
        cfms(s, W[(size_t)k * n + r], t2[k]);
      }
      y[r] = s;
      if (r > j + 1) ss += s.x * s.x + s.y * s.y;
    }
    ss = block_sum(ss, scratch);  // contains the barrier that publishes y[]
    if (t == 0) d[(size_t)z * n + j] = y[j].x;
    if (j + 1 < n) {
      const cplx al = y[j + 1];
      cplx tau, scale;
      double beta;
      if (ss == 0.0 && al.y == 0.0) {
        tau = cmake(0.0, 0.0);
        scale = cmake(0.0, 0.0);
        beta = al.x;
      } else {
        beta = -copysign(sqrt(al.x * al.x + al.y * al.y + ss), al.x);
        tau = cmake((beta - al.x) / beta, -al.y / beta);
        const double dr = al.x - beta, di = al.y, den = 1.0 / (dr * dr + di * di);
        scale = cmake(dr * den, -di * den);  // 1 / (alpha - beta)
      }
      if (t == 0) {
        e[(size_t)z * n + j] = beta;
        scal[2 * z] = tau.x;
        scal[2 * z + 1] = tau.y;
      }
      for (int r = j + 1 + t; r < n; r += PT) {
        const cplx vv = (r == j + 1) ? cmake(1.0, 0.0) : cmul(y[r], scale);
        V[(size_t)i * n + r] = vv;
        V2[(size_t)i * n + r] = vv;
      }
    }
  }
}
}  // namespace


size_t tridiag_vw_elems(int n, int nb) { return (size_t)3 * nb * n; }
size_t tridiag_p_elems(int n) {
  const size_t nblk = (n + TS - 1) / TS;
  return nblk * nblk * TS;
}

// Host driver: all matrices of the batch advance in lock step, two launches per column and one zgemm per panel.
int launch_tridiag(int n, int lda, int nb, BatchRef A, BatchRef VW, BatchRef P, double *d, double *e, double *scal,
                   int ncells, int inner, cudaStream_t s) {
  int launches = 0;
  const int nmat = ncells * inner;
  const int nblk = (n + TS - 1) / TS;
  if (nb > 32) nb = 32;
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(hemv_kernel, (int)kHemvSmem, attr_mask);
  for (int j0 = 0; j0 < n; j0 += nb) {
    const int pn = n - j0 < nb ? n - j0 : nb;
    for (int i = 0; i < pn; ++i) {
      const int j = j0 + i;
      // finish of the previous column of this panel (if any) fused with the reflector of column j
      const int ifin = i > 0 ? i - 1 : -1;
      const int tb0_fin = ifin >= 0 ? (j0 + ifin + 1) / TS : 0;
      { KScope ks(KC_PANEL, 0.0, s);
        panel_step_kernel<<<nmat, PT, 0, s>>>(n, lda, nb, j0, ifin, i, tb0_fin, nblk, A, VW, P, d, e, scal, inner); }
      ++launches;
      if (j + 1 < n) {
        const int tb0 = (j + 1) / TS, nt = nblk - tb0;
        const double m = n - j - 1;
        KScope ks(KC_HEMV, 8.0 * m * (m + 1.0) * nmat, s);  // bytes of the lower triangle read once
        hemv_kernel<<<dim3(nt, nt, nmat), NT, kHemvSmem, s>>>(n, lda, j, tb0, nblk, A, VW, i, P, inner);
        ++launches;
      }
    }
    const int jlast = j0 + pn - 1;
    const int rem = n - j0 - pn;
    if (rem <= 0) break;  // the last column has no reflector and nothing trails it
    panel_step_kernel<<<nmat, PT, 0, s>>>(n, lda, nb, j0, pn - 1, -1, (jlast + 1) / TS, nblk, A, VW, P, d, e, scal, inner);
    ++launches;
    // A22 -= [V W] [W V]^H on the lower tiles
    GemmDesc g{};
    g.ncells = ncells; g.inner = inner; g.kclass = KC_GEMM_TRIDIAG;
    g.M = rem; g.N = rem; g.K = 2 * nb; g.opA = 0; g.opB = 1;
    g.A = VW; g.A.off += j0 + pn; g.lda = n;
    g.B = VW; g.B.off += (long long)nb * n + j0 + pn; g.ldb = n;
    g.C = A; g.C.off += (long long)(j0 + pn) * (lda + 1); g.ldc = lda;
    g.alpha = cmake(-1.0, 0.0); g.beta = cmake(1.0, 0.0); g.flags = BS_GEMM_LOWER_ONLY;
    launch_zgemm(g, s);
    ++launches;
  }
  return launches;
}

}  // namespace bsk
