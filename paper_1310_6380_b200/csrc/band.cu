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
// Workspace per matrix (VW): six slots of n x b complex; SM: coefficient blocks, tau and the split-K partial products.
//
// Band widths <= 16 take the panels in PAIRS (launch_sy2sb): the trailing matrix is read and written once per 2b columns
// by one rank-4b update (K = 4b = 64 at b = 16: the k-loop length of the b = 32 reduction) instead of twice by rank-2b
// updates.  Panel 2 of a pair is factored after only ITS b columns have received panel 1's update (a look-ahead of width
// b), and its Z = A22'' V2 with the not yet updated trailing matrix A22 is corrected by small products:
//   A22'' = A22 - V1 X1^H - X1 V1^H   =>   Z2 = A22 V2 - V1 (X1^H V2) - X1 (V1^H V2) = Z0 - V1 W1 - X1 W2,
//   S = V2^H Z2 = S0 - W2^H W1 - W1^H W2,   X2 = Z2 T2 + V2 M2 = [V1 V2 X1 Z0] [-W1 T2; M2; -W2 T2; T2]   (one GEMM, K = 4b),
//   A22[b:, b:] -= [V1 V2 X1 X2] [X1 X2 V1 V2]^H   (slots 0..3 times slots 2..5: V1 V2 X1 X2 V1 V2).
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int KS = 8;         // largest split-K factor of the Gram product [G | S] = V^H [V | Z] (one output tile per matrix)
// The factor actually used depends on the number of rows only (never on the batch: a matrix gets the same bits alone and
// in a batch): a tall product needs the parallelism, a short one only pays for writing and re-reading the partials
// (C4, m <= 226: 128 KB per matrix and panel, 20 GB per step with KS = 8).
inline int ksplit_of(int m) { return m >= 1024 ? 8 : (m >= 512 ? 4 : (m >= 256 ? 2 : 1)); }

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
  if (K == 1) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
    if (lane == 0) red[warp * K] = v[0];
  } else {
    // first level, transposed: at the stage with partner distance 16, 8, ... a lane keeps half of its values and receives
    // the partner's partial sums of those (KP/2 + KP/4 + ... exchanges instead of 5 KP); a kept sum is own + partner, the
    // butterfly's own operation in the same stage order, so the totals have the butterfly's bits.  Lane bit 4 - s chooses at
    // stage s: the lane ends with value own = bit4 + 2 bit3 + ...
    constexpr int KP = K <= 2 ? 2 : (K <= 4 ? 4 : (K <= 8 ? 8 : 16));
    static_assert(K <= 16, "");
    double w[KP];
#pragma unroll
    for (int k = 0; k < KP; ++k) w[k] = k < K ? v[k] : 0.0;
    int own = 0;
#pragma unroll
    for (int st = 0; st < 5; ++st) {
      const int o = 16 >> st, cnt = KP >> (st + 1);
      if (cnt >= 1) {
        const int bit = (lane >> (4 - st)) & 1;
#pragma unroll
        for (int q = 0; q < cnt; ++q) {
          const double keep = bit ? w[2 * q + 1] : w[2 * q], send = bit ? w[2 * q] : w[2 * q + 1];
          w[q] = keep + __shfl_xor_sync(0xffffffffu, send, o);
        }
        own += bit << st;
      } else {
        w[0] += __shfl_xor_sync(0xffffffffu, w[0], o);
      }
    }
    if ((lane & (32 / KP - 1)) == 0 && own < K) red[warp * K + own] = w[0];
  }
  __syncthreads();
  // second level: value k by warp k mod (number of warps), not all K of them one after the other by warp 0 (the same
  // butterfly over the same numbers: same bits)
  for (int k = warp; k < K; k += NTHR / 32) {
    double x = lane < NTHR / 32 ? red[lane * K + k] : 0.0;
    // (with W < 32 warps the stages at distance >= W add exact zeros to the lanes that matter: skipped, same bits)
#pragma unroll
    for (int o = (NTHR / 32 < 32 ? NTHR / 32 : 32) / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane == 0) res[k] = x;
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
                                                        int inner, int slot1, int slot2) {
  extern __shared__ __align__(16) unsigned char qr_smem[];
  const int r0 = c0 + b, m = n - r0;
  cplx *sp = reinterpret_cast<cplx *>(qr_smem);                 // [SW][m]
  double *red = reinterpret_cast<double *>(sp + (size_t)SW * m);  // [NTHR/32][32]
  double *res = red + (NTHR / 32) * 32;                           // [32]
  cplx *scal = reinterpret_cast<cplx *>(res + 32);                // tau, scale, then T (SW x SW)
  cplx *Tm = scal + 2;
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *Ag = batch_ptr(A, cell, mi);
  cplx *V1 = batch_ptr(VW, cell, mi) + (size_t)slot1 * b * n;  // the two copies of V: slots (n x b each) of the workspace
  cplx *V2 = batch_ptr(VW, cell, mi) + (size_t)slot2 * b * n;
  double *tau_out = reinterpret_cast<double *>(batch_ptr(SM, cell, mi) + (size_t)4 * b * b);
  const int kq = min(b, m - 1);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

  for (int js = 0; js < b; js += SW) {
    // 1. sub-panel -> shared memory
#pragma unroll
    for (int jj = 0; jj < SW; ++jj)  // (column by column: no integer division per element)
      for (int i = t; i < m; i += NTHR) sp[(size_t)jj * m + i] = Ag[(size_t)(r0 + i) + (size_t)(c0 + js + jj) * lda];
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
          // norm and reciprocals by rsqrt / rcp.approx + Newton steps (each good to about 1 ulp) instead of the IEEE square
          // root and three divisions: the whole CTA waits for this thread at the next barrier, once per column
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
        // (every loop fully unrolled: Gm, Tl and taus stay in registers; with run-time indices they lived in local memory
        // and this 4 x 4 recurrence alone took 12 % of the kernel)
        cplx Gm[SW][SW];
        {
          int e = 0;
#pragma unroll
          for (int a = 0; a < SW; ++a)
#pragma unroll
            for (int c = a + 1; c < SW; ++c) { Gm[a][c] = cmake(gv[2 * e], gv[2 * e + 1]); ++e; }
        }
        // T is built in place in shared memory (row-major Tm[a * SW + c]; this thread reads back only what it wrote):
        // the 64-register variants have no room for a second 4 x 4 complex array next to Gm
#pragma unroll
        for (int a = 0; a < SW; ++a)
#pragma unroll
          for (int c = 0; c < SW; ++c) Tm[a * SW + c] = cmake(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < SW; ++c) {
          Tm[c * SW + c] = taus[c];
#pragma unroll
          for (int a = 0; a < SW; ++a) {
            if (a < c) {
              cplx acc = cmake(0.0, 0.0);
#pragma unroll
              for (int l2 = 0; l2 < SW; ++l2)
                if (l2 >= a && l2 < c) cfma(acc, Tm[a * SW + l2], Gm[l2][c]);
              Tm[a * SW + c] = cmul(cmake(-taus[c].x, -taus[c].y), acc);
            }
          }
        }
      }
    }
    // 4. V columns out
#pragma unroll
    for (int jj = 0; jj < SW; ++jj)
      for (int i = t; i < m; i += NTHR) {
        const cplx v = sp[(size_t)jj * m + i];
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
      {
        // the 2 SW lane sums: transposed reduction (4 + 2 + 1 + 1 + 1 exchanges instead of 40; a kept sum is own + partner
        // in the butterfly's stage order: same bits), then every total is broadcast from the lane that holds it
        double w[2 * SW];
#pragma unroll
        for (int k = 0; k < SW; ++k) { w[2 * k] = d[k].x; w[2 * k + 1] = d[k].y; }
#pragma unroll
        for (int st = 0; st < 5; ++st) {
          const int o = 16 >> st, cnt = (2 * SW) >> (st + 1);
          if (cnt >= 1) {
            const int bit = (lane >> (4 - st)) & 1;
#pragma unroll
            for (int q = 0; q < cnt; ++q) {
              const double keep = bit ? w[2 * q + 1] : w[2 * q], send = bit ? w[2 * q] : w[2 * q + 1];
              w[q] = keep + __shfl_xor_sync(0xffffffffu, send, o);
            }
          } else {
            w[0] += __shfl_xor_sync(0xffffffffu, w[0], o);
          }
        }
        // value e = b0 + 2 b1 + 4 b2 lives in the lanes with bit 4 = b0, bit 3 = b1, bit 2 = b2
#pragma unroll
        for (int e = 0; e < 2 * SW; ++e) {
          const int src = ((e & 1) << 4) | (((e >> 1) & 1) << 3) | (((e >> 2) & 1) << 2);
          const double tot = __shfl_sync(0xffffffffu, w[0], src);
          if (e & 1) d[e >> 1].y = tot; else d[e >> 1].x = tot;
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
__global__ void __launch_bounds__(1024) wy_small_kernel(int b, BatchRef SM, int inner, int ks) {
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
    for (int k = 0; k < ks; ++k) {  // fixed order: deterministic
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

// Second panel of a pair (see the header): from the split-K partials of Gm = [V1 V2 X1]^H [V2 X1 Z0] (3b x 3b, ld 3b) and
// tau of panel 2, the coefficient block Cf (4b x b, ld 4b) of  X2 = [V1 V2 X1 Z0] Cf :
//   W2 = V1^H V2 = Gm[0:b, 0:b],  G = V2^H V2 = Gm[b:2b, 0:b],  W1 = X1^H V2 = Gm[2b:3b, 0:b],  S0 = V2^H Z0 = Gm[b:2b, 2b:3b],
//   S = S0 - W2^H W1 - W1^H W2,  T2 as in wy_small_kernel,  M2 = -1/2 T2^H S T2,  Cf = [-W1 T2; M2; -W2 T2; T2].
// SM per matrix: Cf at 0; tau at 4 b^2; partials at 4 b^2 + 64.
__global__ void __launch_bounds__(1024) wy_pair_kernel(int b, BatchRef SM, int inner, int ks) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *T = reinterpret_cast<cplx *>(smem_raw);  // b x b, T[i + j*b]
  cplx *S = T + b * b;
  cplx *U = S + b * b;
  cplx *G = U + b * b;
  cplx *W1 = G + b * b;
  cplx *W2 = W1 + b * b;
  cplx *taus = W2 + b * b;
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *sm = batch_ptr(SM, cell, mi);
  const cplx *part = sm + (size_t)4 * b * b + 64;
  cplx *out = sm;
  const int t = threadIdx.x, b3 = 3 * b;
  if (t < b) taus[t] = sm[(size_t)4 * b * b + t];
  auto gm = [&](int r, int c) {  // fixed order over the k-splits: deterministic
    cplx a = cmake(0.0, 0.0);
    for (int k = 0; k < ks; ++k) a = cadd(a, part[(size_t)k * b3 * b3 + r + (size_t)c * b3]);
    return a;
  };
  for (int i = t; i < b * b; i += blockDim.x) {
    const int r = i % b, c = i / b;
    W2[i] = gm(r, c);
    G[i] = gm(b + r, c);
    W1[i] = gm(2 * b + r, c);
    S[i] = gm(b + r, 2 * b + c);
    T[i] = cmake(0.0, 0.0);
    U[i] = (r == c) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
  }
  __syncthreads();
  for (int i = t; i < b * b; i += blockDim.x) {  // S = S0 - W2^H W1 - W1^H W2
    const int r = i % b, c = i / b;
    cplx a = S[i];
    for (int l = 0; l < b; ++l) {
      cplx p = cmake(0.0, 0.0);
      cfmac(p, W2[l + r * b], W1[l + c * b]);
      cfmac(p, W1[l + r * b], W2[l + c * b]);
      a = csub(a, p);
    }
    S[i] = a;
  }
  __syncthreads();
  for (int l = b - 1; l >= 0; --l) {  // T2: column-oriented back substitution, as in wy_small_kernel
    const cplx tl = taus[l];
    for (int e = t; e < b * b; e += blockDim.x) {
      const int i = e % b, j = e / b;
      if (j < l || i > l) continue;
      const cplx x = cmul(tl, U[l + j * b]);
      if (i == l) T[e] = x;
      else { cplx r = U[e]; cfms(r, G[i + l * b], x); U[e] = r; }
    }
    __syncthreads();
  }
  for (int i = t; i < b * b; i += blockDim.x) {  // U = S T
    const int r = i % b, c = i / b;
    cplx acc = cmake(0.0, 0.0);
    for (int l = 0; l <= c; ++l) cfma(acc, S[r + l * b], T[l + c * b]);
    U[i] = acc;
  }
  __syncthreads();
  for (int i = t; i < b * b; i += blockDim.x) {
    const int r = i % b, c = i / b;
    cplx m2 = cmake(0.0, 0.0), a1 = cmake(0.0, 0.0), a2 = cmake(0.0, 0.0);
    for (int l = 0; l <= r; ++l) cfmac(m2, T[l + r * b], U[l + c * b]);   // (T^H U)[r, c]
    for (int l = 0; l <= c; ++l) {                                         // (W T)[r, c], T upper triangular
      cfma(a1, W1[r + l * b], T[l + c * b]);
      cfma(a2, W2[r + l * b], T[l + c * b]);
    }
    cplx *col = out + (size_t)c * 4 * b;
    col[r] = cmake(-a1.x, -a1.y);
    col[b + r] = cscale(m2, -0.5);
    col[2 * b + r] = cmake(-a2.x, -a2.y);
    col[3 * b + r] = T[i];
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

size_t band_vw_elems(int n, int b) { return (size_t)6 * b * n; }
size_t band_sm_elems(int b) { return (size_t)4 * b * b + 64 + (size_t)KS * 9 * b * b; }
size_t band_ab_elems(int n, int b) { return (size_t)n * 2 * b; }

// Stage 1 for every matrix of the batch in lock step; on exit AB holds the band (ldab = 2b, bulge space zeroed).
int launch_sy2sb(int n, int lda, int b, BatchRef A, BatchRef VW, BatchRef SM, BatchRef AB, int ncells, int inner,
                 cudaStream_t s, const BatchRef *keepV, const BatchRef *keepT) {
  int launches = 0;
  const int nmat = ncells * inner;
  static unsigned long long m1 = 0, m2 = 0, m3 = 0, m4 = 0, m5 = 0;
  ensure_dyn_smem(panel_qr_kernel<1024>, 140 * 1024, m1);
  ensure_dyn_smem(panel_qr_kernel<256, 2>, 48 * 1024, m2);
  ensure_dyn_smem(panel_qr_kernel<256, 4>, 48 * 1024, m3);
  ensure_dyn_smem(wy_small_kernel, (4 * 32 * 32 + 32) * (int)sizeof(cplx), m4);
  ensure_dyn_smem(wy_pair_kernel, (6 * 32 * 32 + 32) * (int)sizeof(cplx), m5);
  auto slot = [&](int k, int r0) { BatchRef r = VW; r.off += (long long)k * b * n + r0; return r; };  // rows r0.. of slot k
  auto qr = [&](int c0, int s1, int s2) {
    const int m = n - (c0 + b);
    KScope ks(KC_PANEL, 0.0, s);
    auto smem_of = [&](int nthr) {
      return (size_t)SW * m * sizeof(cplx) + (nthr + 32) * sizeof(double) + (2 + SW * SW) * sizeof(cplx);
    };
    // The thread count depends on m only (it decides the summation order, i.e. the bits); the register budget (CTAs per SM)
    // on the batch.  m <= 256: 128 threads (at most two rows per thread, four warps per block reduction) and twice as many
    // CTAs per SM: C4 panel 15.2 -> 11.2 ms (64 threads: 10.5 ms there, but C2 1.22 -> 1.51 and C3 3.40 -> 3.68 ms; 128
    // threads: 1.29 and 3.47).
    if (m > 640) panel_qr_kernel<1024><<<nmat, 1024, smem_of(1024), s>>>(n, lda, b, c0, A, VW, SM, inner, s1, s2);
    else if (m > 256 && nmat > 592) panel_qr_kernel<256, 4><<<nmat, 256, smem_of(256), s>>>(n, lda, b, c0, A, VW, SM, inner, s1, s2);
    else if (m > 256) panel_qr_kernel<256, 2><<<nmat, 256, smem_of(256), s>>>(n, lda, b, c0, A, VW, SM, inner, s1, s2);
    else if (nmat > 592) panel_qr_kernel<128, 8><<<nmat, 128, smem_of(128), s>>>(n, lda, b, c0, A, VW, SM, inner, s1, s2);
    else panel_qr_kernel<128, 4><<<nmat, 128, smem_of(128), s>>>(n, lda, b, c0, A, VW, SM, inner, s1, s2);
    ++launches;
  };
  auto gemm = [&](int kclass, int M, int N, int K, int opA, int opB, int flags, BatchRef Ar, int la, BatchRef Br, int lb,
                  BatchRef Cr, int lc, double alpha, double beta, int ksplit = 0, long long sstride = 0) {
    GemmDesc g{};
    g.ncells = ncells; g.inner = inner; g.kclass = kclass;
    g.M = M; g.N = N; g.K = K; g.opA = opA; g.opB = opB; g.flags = flags;
    g.A = Ar; g.lda = la; g.B = Br; g.ldb = lb; g.C = Cr; g.ldc = lc;
    g.alpha = cmake(alpha, 0.0); g.beta = cmake(beta, 0.0);
    g.ksplit = ksplit; g.split_stride = sstride;
    launch_zgemm(g, s); ++launches;
  };
  auto keep = [&](int c0, int vslot, long long t_off, int t_ld) {  // mode shapes: V and T of this panel are needed again
    if (!keepV) return;
    const int r0 = c0 + b, m = n - r0;
    BatchRef dst = *keepV;
    dst.off += (long long)c0 * n + r0;
    launch_copy_matrix(m, b, slot(vslot, r0), n, dst, n, ncells, inner, s); ++launches;
    BatchRef src = SM;
    src.off += t_off;
    dst = *keepT; dst.off += (long long)(c0 / b) * b * b;
    launch_copy_matrix(b, b, src, t_ld, dst, b, ncells, inner, s); ++launches;
  };
  auto trailing = [&](int r0) { BatchRef r = A; r.off += (long long)r0 * (lda + 1); return r; };
  BatchRef smG = SM, smOut = SM, smCf = SM;
  smG.off += (long long)4 * b * b + 64;  // split-K partials
  smOut.off += (long long)2 * b * b;     // [M2; T] of a single panel (ld 2b)
  // One panel: V -> slots (sv, sv2), Z -> slot sv2 + 1, X -> slot sx;  Gram with B = [V copy | Z], X = [V copy | Z] [M2; T]
  auto single_front = [&](int c0, int sv, int sv2, int sx) {
    const int r0 = c0 + b, m = n - r0;
    qr(c0, sv, sv2);
    gemm(KC_GEMM_HEMM, m, b, m, 0, 0, BS_GEMM_A_HERM_LOWER, trailing(r0), lda, slot(sv, r0), n, slot(sv2 + 1, r0), n, 1.0, 0.0);
    gemm(KC_GEMM_WY, b, 2 * b, m, 1, 0, 0, slot(sv, r0), n, slot(sv2, r0), n, smG, b, 1.0, 0.0, ksplit_of(m), (long long)2 * b * b);
    {
      KScope ks(KC_OTHER, 0.0, s);
      // few matrices: one thread per entry (latency); many: smaller CTAs, several per SM (throughput; C4: 256 threads 3.98 ms of
      // `other` per step, 128: 3.31, 64: 3.44, 32: 4.68).  Every entry is summed by one thread: the thread count changes no bit
      wy_small_kernel<<<nmat, nmat > 592 ? 128 : b * b, (4 * b * b + b) * sizeof(cplx), s>>>(b, SM, inner, ksplit_of(m));
      ++launches;
    }
    keep(c0, sv, (long long)2 * b * b + b, 2 * b);
    gemm(KC_GEMM_WY, m, b, 2 * b, 0, 0, 0, slot(sv2, r0), n, smOut, 2 * b, slot(sx, r0), n, 1.0, 0.0);
  };
  int c0 = 0;
  // Pairs pay off where the trailing updates dominate: measured S6 totals (ms, pairs / single panels) C5 (n = 1922) 235.7 /
  // 249.8, C3 (n = 882) 32.1 / 31.5, C2 (n = 450) 8.3 / 7.8, C4 (n = 242, 10240 matrices) 155 / 141 (the extra small products).
  // The rule depends on n only, so a batch and its members take the same path.  (The in-place X2 product needs one column
  // tile: N = b <= 16.)
  const bool pairs = b <= 16 && n >= 1200;
  while (c0 + b < n - 1) {
    const int r0 = c0 + b, m = n - r0;  // m >= 2
    const bool second = pairs && (c0 + 2 * b < n - 1);
    if (!second) {
      // a single panel: slots [. V X V Z .]: A22 -= [V | X] [X | V]^H on the lower tiles
      single_front(c0, 1, 3, 2);
      gemm(KC_GEMM_TRIDIAG, m, m, 2 * b, 0, 1, BS_GEMM_LOWER_ONLY, slot(1, r0), n, slot(2, r0), n, trailing(r0), lda, -1.0, 1.0);
      c0 += b;
      continue;
    }
    // ---- a pair of panels: slots [V1 V2 X1 X2 V1 V2]
    single_front(c0, 0, 4, 2);  // V1 -> 0 and 4, Z1 -> 5, X1 -> 2
    // look-ahead: only the next panel's b columns receive panel 1's update now:  A[r0:, r0:r0+b] -= X1 V1[0:b]^H + V1 X1[0:b]^H
    gemm(KC_GEMM_TRIDIAG, m, b, b, 0, 1, 0, slot(2, r0), n, slot(0, r0), n, trailing(r0), lda, -1.0, 1.0);
    gemm(KC_GEMM_TRIDIAG, m, b, b, 0, 1, 0, slot(4, r0), n, slot(2, r0), n, trailing(r0), lda, -1.0, 1.0);
    const int c1 = c0 + b, r1 = c1 + b, m2 = n - r1;
    qr(c1, 1, 5);  // V2 -> 1 and 5
    // Z0 = A22 V2 with the trailing matrix as it was before panel 1's update -> slot 3
    gemm(KC_GEMM_HEMM, m2, b, m2, 0, 0, BS_GEMM_A_HERM_LOWER, trailing(r1), lda, slot(1, r1), n, slot(3, r1), n, 1.0, 0.0);
    // Gm = [V1 V2 X1]^H [V2 X1 Z0]  (3b x 3b, split-K)
    gemm(KC_GEMM_WY, 3 * b, 3 * b, m2, 1, 0, 0, slot(0, r1), n, slot(1, r1), n, smG, 3 * b, 1.0, 0.0, ksplit_of(m2), (long long)9 * b * b);
    {
      KScope ks(KC_OTHER, 0.0, s);
      wy_pair_kernel<<<nmat, nmat > 592 ? 256 : b * b, (6 * b * b + b) * sizeof(cplx), s>>>(b, SM, inner, ksplit_of(m2));
      ++launches;
    }
    keep(c1, 1, (long long)3 * b, 4 * b);
    // X2 = [V1 V2 X1 Z0] Cf, written over Z0 (slot 3): a CTA of the 64 x 16 tiling owns complete rows and has read all of
    // its A operand before its epilogue stores
    gemm(KC_GEMM_WY, m2, b, 4 * b, 0, 0, 0, slot(0, r1), n, smCf, 4 * b, slot(3, r1), n, 1.0, 0.0);
    // A22[b:, b:] -= [V1 V2 X1 X2] [X1 X2 V1 V2]^H on the lower tiles: ONE read-modify-write of the trailing matrix per pair
    gemm(KC_GEMM_TRIDIAG, m2, m2, 4 * b, 0, 1, BS_GEMM_LOWER_ONLY, slot(0, r1), n, slot(2, r1), n, trailing(r1), lda, -1.0, 1.0);
    c0 += 2 * b;
  }
  {
    KScope ks(KC_OTHER, 0.0, s);
    band_extract_kernel<<<dim3((n + 7) / 8, 1, nmat), 256, 0, s>>>(n, lda, b, 2 * b, A, AB, inner);
    ++launches;
  }
  return launches;
}

}  // namespace bsk
