// Batched complex128 GEMM on the FP64 tensor pipe (mma.sync m8n8k4 f64 -> DMMA on sm_100a; tcgen05 has no f64 kind).
// C = alpha op(A) op(B) + beta C, column-major interleaved complex, (re,im) kept interleaved in shared memory (one
// LDS.128 fetches both).  The complex product is taken in its "3M" form, three real DMMAs per complex multiply-add
// instead of four:  Re = ar br - ai bi,  Im = (ar + ai)(br + bi) - ar br - ai bi  (norm-wise backward stable; the
// tolerance budget is in DESIGN.md section 5, zgemm).
#include "bs_internal.cuh"
#include <type_traits>

namespace bsk {

namespace {
// CTA tile BM x BN = 32 x 32, four warps of 16 x 16 each (three accumulator sets of 2 x 2 m8n8 tiles = 48 registers),
// four CTAs per SM: small CTAs in different phases hide each other's prologue and read-modify-write epilogue, which
// is what the K = 2b = 64 rank-2b updates consist of.  Row strides are padded by 2 (conflict-free fragments).
template <int BM, int BN, int BK, int STAGES>
constexpr size_t smem_bytes() { return (size_t)STAGES * BK * ((BM + 2) + (BN + 2)) * sizeof(cplx); }

__device__ __forceinline__ void cp16(unsigned dst, const void *src, bool ok) {  // dst: shared-space address
  const int sz = ok ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// HERM = 1: A is an M x M Hermitian matrix of which only the LOWER triangle is valid (K == M, OPA == 0):
//   op(A)[m][k] = A[m][k] for m > k, Re A[m][m] for m == k, conj(A[k][m]) for m < k  (the HEMM of the band reduction).
template <int OPA, int OPB, int HERM, int BM, int BN, int NT, int MI, int BK, int STAGES, int CPS>
__global__ void __launch_bounds__(NT, CPS) zgemm_kernel(const GemmDesc g) {
  constexpr int NI = 2;                                              // 8-column sub-tiles per warp
  constexpr int LDA_S = BM + 2, LDB_S = BN + 2, WMN = BM / (8 * MI);  // WMN warps along m, (NT / 32) / WMN along n
  static_assert((BM / (8 * MI)) * (BN / (8 * NI)) == NT / 32, "warps of 8 MI x 8 NI");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx(*As)[BK][LDA_S] = reinterpret_cast<cplx(*)[BK][LDA_S]>(smem_raw);
  cplx(*Bs)[BK][LDB_S] = reinterpret_cast<cplx(*)[BK][LDB_S]>(smem_raw + (size_t)STAGES * BK * LDA_S * sizeof(cplx));

  // grid.x = (M tiles) x (matrices x k-splits): grid.z is limited to 65535, the batch of config 4 is not
  const int tiles_m = (g.M + BM - 1) / BM;
  int bz, m0, n0;
  if (g.flags & BS_GEMM_LOWER_ONLY) {
    // only the tiles of the lower triangle are launched: with R = BM / BN column tiles per row tile,
    // tile t -> (i, j), j < R (i + 1), t = R i (i + 1) / 2 + j
    constexpr int R = BM / BN;
    const int ntri = R * tiles_m * (tiles_m + 1) / 2;
    bz = blockIdx.x / ntri;
    const int tix = blockIdx.x % ntri;
    int i = (int)((sqrtf(8.0f * (float)(tix / R) + 1.0f) - 1.0f) * 0.5f);
    while (R * i * (i + 1) / 2 > tix) --i;
    while (R * (i + 1) * (i + 2) / 2 <= tix) ++i;
    m0 = i * BM;
    n0 = (tix - R * i * (i + 1) / 2) * BN;
  } else {
    bz = blockIdx.x / tiles_m;
    m0 = (blockIdx.x % tiles_m) * BM;
    n0 = blockIdx.y * BN;
  }
  if ((g.flags & BS_GEMM_LOWER_ONLY) && n0 >= m0 + BM) return;
  const int nsplit = g.ksplit > 1 ? g.ksplit : 1;
  const int ks = bz % nsplit, zz = bz / nsplit;
  const int cell = zz / g.inner, bi = zz % g.inner;
  const cplx *__restrict__ A = batch_ptr(g.A, cell, bi);
  const cplx *__restrict__ B = batch_ptr(g.B, cell, bi);
  cplx *C = batch_ptr(g.C, cell, bi) + (size_t)ks * g.split_stride;

  int klo = 0, khi = g.K;
  if (nsplit > 1) {
    const int kc = ((g.K + nsplit - 1) / nsplit + BK - 1) / BK * BK;
    klo = ks * kc;
    khi = min(g.K, klo + kc);
  }
  if (g.flags & BS_GEMM_KLO_ROW) klo = max(klo, m0);
  if (g.flags & BS_GEMM_KHI_ROW) khi = min(khi, m0 + BM);
  if (g.flags & BS_GEMM_KLO_COL) klo = max(klo, n0);
  if (g.flags & BS_GEMM_KHI_COL) khi = min(khi, n0 + BN);
  klo &= ~(BK - 1);
  const int nkt = khi > klo ? (khi - klo + BK - 1) / BK : 0;

  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int wm = warp % WMN, wn = warp / WMN;  // warp tile 16 x 32

  // Per-thread load slots: RA + RB 16-byte elements per k-tile.  Source pointers are set up once and advanced by a
  // constant per k-tile (load_tile is called for kt = 0, 1, 2, ... in order); the address arithmetic of a k-tile is a
  // few instructions, not a chain in front of the tensor work.  HERM keeps two sets for A: the direct one for k-tiles
  // below the diagonal, the transposed one above it; the few k-tiles that cross it compute their addresses in place.
  constexpr int RA = BM * BK / NT, RB = (BN * BK + NT - 1) / NT;
  static_assert(RA >= 1, "A slots");
  constexpr bool TRA = OPA != 0;  // the only set reads transposed positions
  const cplx *pa[RA], *pat[HERM ? RA : 1], *pb[RB];
  int ka[RA], kat[HERM ? RA : 1], kb[RB];
  bool va[RA], vat[HERM ? RA : 1], vb[RB];
  unsigned sa[RA], sat[HERM ? RA : 1], sb[RB];
  const unsigned as_base = (unsigned)__cvta_generic_to_shared(&As[0][0][0]);
  const unsigned bs_base = (unsigned)__cvta_generic_to_shared(&Bs[0][0][0]);
#pragma unroll
  for (int r = 0; r < RA; ++r) {
    int m, k;
    if (!TRA) { m = t % BM; k = t / BM + (NT / BM) * r; } else { k = t % BK; m = t / BK + (NT / BK) * r; }
    ka[r] = k; va[r] = m0 + m < g.M; sa[r] = as_base + (unsigned)((k * LDA_S + m) * sizeof(cplx));
    pa[r] = !TRA ? A + (size_t)(m0 + m) + (size_t)(klo + k) * g.lda : A + (size_t)(klo + k) + (size_t)(m0 + m) * g.lda;
    if (HERM) {
      k = t % BK; m = t / BK + (NT / BK) * r;
      kat[r] = k; vat[r] = m0 + m < g.M; sat[r] = as_base + (unsigned)((k * LDA_S + m) * sizeof(cplx));
      pat[r] = A + (size_t)(klo + k) + (size_t)(m0 + m) * g.lda;
    }
  }
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    int n, k;
    if (OPB == 0) { k = t % BK; n = t / BK + (NT / BK) * r; } else { n = t % BN; k = t / BN + (NT / BN) * r; }
    kb[r] = k; vb[r] = (n0 + n < g.N) && !(BN * BK < NT && t >= BN * BK);
    sb[r] = bs_base + (unsigned)((k * LDB_S + n) * sizeof(cplx));
    pb[r] = OPB == 0 ? B + (size_t)(klo + k) + (size_t)(n0 + n) * g.ldb : B + (size_t)(n0 + n) + (size_t)(klo + k) * g.ldb;
  }
  const size_t step_a = !TRA ? (size_t)BK * g.lda : (size_t)BK, step_b = OPB == 0 ? (size_t)BK : (size_t)BK * g.ldb;
  auto load_tile = [&](int kt, int stage) {
    const int k0 = klo + kt * BK;
    const unsigned oa = (unsigned)(stage * BK * LDA_S * sizeof(cplx)), ob = (unsigned)(stage * BK * LDB_S * sizeof(cplx));
    const bool above = HERM && k0 >= m0 + BM - 1;                 // the whole k-tile lies above the diagonal
    const bool cross = HERM && !above && k0 + BK - 1 > m0;        // it crosses the diagonal: per element
#pragma unroll
    for (int r = 0; r < RA; ++r) {
      if (cross) {
        const int m = t % BM, k = t / BM + (NT / BM) * r;
        const bool tr = k0 + k > m0 + m, ok = (m0 + m < g.M) && (k0 + k < khi);
        const cplx *src = !tr ? A + (size_t)(m0 + m) + (size_t)(k0 + k) * g.lda
                              : A + (size_t)(k0 + k) + (size_t)(m0 + m) * g.lda;
        cp16(sa[r] + oa, ok ? src : A, ok);
      } else if (above) {
        const bool ok = vat[r] && (k0 + kat[r] < khi);
        cp16(sat[r] + oa, ok ? pat[r] : A, ok);
      } else {
        const bool ok = va[r] && (k0 + ka[r] < khi);
        cp16(sa[r] + oa, ok ? pa[r] : A, ok);
      }
      pa[r] += step_a;
      if (HERM) pat[r] += BK;
    }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const bool ok = vb[r] && (k0 + kb[r] < khi);
      cp16(sb[r] + ob, ok ? pb[r] : B, ok);
      pb[r] += step_b;
    }
  };

  // beta != 0: the C tile is read only in the epilogue; warm it into L2 now so that the read-modify-write does not
  // pay DRAM latency after the (short, K = 2b) main loop of the rank-2b updates
  // (beta == 1 needs neither: the update goes out as reductions, see the epilogue)
  const bool accumulate = g.beta.x == 1.0 && g.beta.y == 0.0;
  if ((g.beta.x != 0.0 || g.beta.y != 0.0) && !accumulate) {
#pragma unroll
    for (int ni = 0; ni < NI; ++ni) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int row = m0 + wm * (8 * MI) + (lane >> 2), col = n0 + wn * (8 * NI) + ni * 8 + (lane & 3) * 2 + j;
        if (row < g.M && col < g.N) asm volatile("prefetch.global.L2 [%0];\n" ::"l"(C + (size_t)row + (size_t)col * g.ldc));
      }
    }
  }
  // c1 = sum ar br, c2 = sum ai bi (stored imaginary parts), c3 = sum (ar +- ai)(br +- bi) (- where conjugated)
  double c1[MI][NI][2], c2[MI][NI][2], c3[MI][NI][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j)
      c1[i][j][0] = c1[i][j][1] = c2[i][j][0] = c2[i][j][1] = c3[i][j][0] = c3[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < nkt) load_tile(s, s);
    cp_commit();
  }
  for (int kt = 0; kt < nkt; ++kt) {
    cp_wait<STAGES - 2>();
    __syncthreads();
    const int st = kt % STAGES;
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      cplx a[MI], b[NI];
#pragma unroll
      for (int mi = 0; mi < MI; ++mi) a[mi] = As[st][kk + (lane & 3)][wm * (8 * MI) + mi * 8 + (lane >> 2)];
#pragma unroll
      for (int ni = 0; ni < NI; ++ni) b[ni] = Bs[st][kk + (lane & 3)][wn * (8 * NI) + ni * 8 + (lane >> 2)];
      if (kk == 0) {  // the fragment loads of this k-tile are in flight: now refill the stage read one k-tile ago
        if (kt + STAGES - 1 < nkt) load_tile(kt + STAGES - 1, (kt + STAGES - 1) % STAGES);
        cp_commit();
      }
      // Conjugations cost no FP64-pipe instruction (the pipe DMMA runs on): a uniform conjugate of A or B only
      // changes signs in the operand sums below and in the epilogue (SGN); the per-element one of HERM flips the
      // sign bit with an integer operation.
      if (HERM) {
#pragma unroll
        for (int mi = 0; mi < MI; ++mi) {
          const int mg = m0 + wm * (8 * MI) + mi * 8 + (lane >> 2), kg = klo + kt * BK + kk + (lane & 3);
          int hi = __double2hiint(a[mi].y), lo = __double2loint(a[mi].y);
          hi = kg > mg ? hi ^ (int)0x80000000 : hi;
          hi = kg == mg ? 0 : hi;
          lo = kg == mg ? 0 : lo;
          a[mi].y = __hiloint2double(hi, lo);
        }
      }
      double bs[NI];
#pragma unroll
      for (int ni = 0; ni < NI; ++ni) bs[ni] = OPB ? b[ni].x - b[ni].y : b[ni].x + b[ni].y;
#pragma unroll
      for (int mi = 0; mi < MI; ++mi) {
        const double as = OPA ? a[mi].x - a[mi].y : a[mi].x + a[mi].y;
#pragma unroll
        for (int ni = 0; ni < NI; ++ni) dmma(c1[mi][ni][0], c1[mi][ni][1], a[mi].x, b[ni].x);
#pragma unroll
        for (int ni = 0; ni < NI; ++ni) dmma(c2[mi][ni][0], c2[mi][ni][1], a[mi].y, b[ni].y);
#pragma unroll
        for (int ni = 0; ni < NI; ++ni) dmma(c3[mi][ni][0], c3[mi][ni][1], as, bs[ni]);
      }
    }
  }
  cp_wait<0>();

  const bool has_beta = (g.beta.x != 0.0 || g.beta.y != 0.0);
  const bool lower = g.flags & BS_GEMM_LOWER_ONLY;
  if (accumulate) {
    // C += alpha A B: every entry receives exactly one addition per launch, sent as two fire-and-forget FP64
    // reductions that L2 performs; no read of C, no latency in the epilogue (deterministic: one addend per entry)
#pragma unroll
    for (int mi = 0; mi < MI; ++mi) {
      const int row = m0 + wm * (8 * MI) + mi * 8 + (lane >> 2);
      if (row >= g.M) continue;
#pragma unroll
      for (int ni = 0; ni < NI; ++ni) {
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const int col = n0 + wn * (8 * NI) + ni * 8 + (lane & 3) * 2 + j;
          if (col >= g.N || (lower && col > row)) continue;
          const double t1 = c1[mi][ni][j], t2 = (OPA != OPB ? -1.0 : 1.0) * c2[mi][ni][j];
          const cplx v = cmul(g.alpha, cmake(t1 - t2, c3[mi][ni][j] - t1 - t2));
          double *dst = reinterpret_cast<double *>(C + (size_t)row + (size_t)col * g.ldc);
          asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(dst), "d"(v.x) : "memory");
          asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(dst + 1), "d"(v.y) : "memory");
        }
      }
    }
    return;
  }
#pragma unroll
  for (int mi = 0; mi < MI; ++mi) {
    const int row = m0 + wm * (8 * MI) + mi * 8 + (lane >> 2);
    if (row >= g.M) continue;
    // all eight C loads of this row first (independent, in flight together), then the eight stores: a load placed
    // after a store to C could not be hoisted above it
    cplx old[NI][2];
#pragma unroll
    for (int ni = 0; ni < NI; ++ni) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int col = n0 + wn * (8 * NI) + ni * 8 + (lane & 3) * 2 + j;
        old[ni][j] = cmake(0.0, 0.0);
        if (has_beta && col < g.N && !(lower && col > row)) old[ni][j] = C[(size_t)row + (size_t)col * g.ldc];
      }
    }
#pragma unroll
    for (int ni = 0; ni < NI; ++ni) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int col = n0 + wn * (8 * NI) + ni * 8 + (lane & 3) * 2 + j;
        if (col >= g.N || (lower && col > row)) continue;
        // c2 holds sum ai bi of the stored imaginary parts: SGN = -1 if exactly one operand is conjugated
        const double t1 = c1[mi][ni][j], t2 = (OPA != OPB ? -1.0 : 1.0) * c2[mi][ni][j];
        cplx v = cmul(g.alpha, cmake(t1 - t2, c3[mi][ni][j] - t1 - t2));
        if (has_beta) v = cadd(v, cmul(g.beta, old[ni][j]));
        C[(size_t)row + (size_t)col * g.ldc] = v;
      }
    }
  }
}

// ---- the Hermitian product of the band reduction, Z = A22 V with exactly 16 columns (band width 16) ---------------
// Same tile shape and accumulators as zgemm_kernel<0, 0, 1, 64, 16, 128>, specialised so that the long parts of the
// k loop carry no per-element logic and the memory side moves every byte once:
//  * k-tiles left of the CTA's diagonal block read A[m][k] down the columns, k-tiles right of it read conj(A[k][m])
//    along the rows of the lower triangle and flip one sign bit per fragment; only the 8 k-tiles of the diagonal
//    block take the per-element path.  Source addresses are one 64-bit base per part plus constant multiples of the
//    column stride; rows beyond M are requested with src-size 0 (zero fill, nothing is read).
//  * Shared-memory layout: tiles read down the columns of A are stored k-major (As[k][m], consecutive lanes write
//    consecutive 16 bytes); tiles read along its rows, and the V tile, are stored m-major (As[m][k ^ 4 (m & 1)]) so
//    that the lanes of a cp.async instruction, which then run along k, again write consecutive shared memory.
//    Measured (profiles/r2_hemm16.md): with lanes along k writing the k-major layout (one row stride per lane) every
//    sector crossed the crossbar twice (8.3 GB instead of 5.3 GB per launch) and the loads alone took 0.85 ms instead
//    of 0.43 ms at m = 1472.
//  * Order of the k-tiles: see block_of below (both readers of a lower-triangle block meet in L2).
// The k order differs from the generic kernel's, so results differ from it in the last bits; they depend only on
// (M, block row), not on the batch.
template <int CPS, int BK, int ST>
__global__ void __launch_bounds__(128, CPS) hemm16_kernel(const GemmDesc g) {
  constexpr int BM = 64, BN = 16, LDA_S = BM + 2, LDB_S = BN + 2;
  static_assert(BK == 8, "the swizzle below is for rows of 8 elements");
  constexpr int STAGE_A = BK * LDA_S, STAGE_B = BN * BK;  // elements; a k-major A tile (BM x BK, row stride BK) fits too
  constexpr int RA = BM * BK / 128, RB = BN * BK / 128, MSTEP = 128 / BK;  // cp.async slots per thread and k-tile
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *As = reinterpret_cast<cplx *>(smem_raw), *Bs = As + ST * STAGE_A;
  const int tiles_m = (g.M + BM - 1) / BM;
  const int zz = blockIdx.x / tiles_m, m0 = (blockIdx.x % tiles_m) * BM;
  const int cell = zz / g.inner, bi = zz % g.inner;
  const cplx *__restrict__ A = batch_ptr(g.A, cell, bi);
  const cplx *__restrict__ B = batch_ptr(g.B, cell, bi);
  cplx *C = batch_ptr(g.C, cell, bi);
  const int M = g.M, nkt = (M + BK - 1) / BK;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5, gq = lane >> 2, tq = lane & 3;

  const unsigned as_s = (unsigned)__cvta_generic_to_shared(As), bs_s = (unsigned)__cvta_generic_to_shared(Bs);
  const long long ldab = (long long)g.lda * (long long)sizeof(cplx);  // bytes per column of A
  // left part: element (m, k) of a k-tile, m = t % 64, k = t / 64 + 2 r
  const int md = t & 63, kd = t >> 6;
  const char *pD = reinterpret_cast<const char *>(A + (m0 + md)) + kd * ldab;
  const unsigned dD = as_s + (unsigned)((kd * LDA_S + md) * sizeof(cplx)), szd = m0 + md < M ? 16u : 0u;
  // right part: k = t % BK, m = t / BK + MSTEP r, read from A[k][m]
  const int km = t % BK, mm = t / BK;
  const char *pM = reinterpret_cast<const char *>(A + km) + (long long)(m0 + mm) * ldab;
  const int swm = (mm & 1) << 2;
  const unsigned dM = as_s + (unsigned)((mm * BK + (km ^ swm)) * sizeof(cplx));
  unsigned szm[RA];
#pragma unroll
  for (int r = 0; r < RA; ++r) szm[r] = m0 + mm + MSTEP * r < M ? 16u : 0u;
  // V: k = t % BK, n = t / BK + MSTEP r
  const long long ldbb = (long long)g.ldb * (long long)sizeof(cplx);
  const char *pB = reinterpret_cast<const char *>(B + km + (size_t)mm * g.ldb);
  const unsigned dB = bs_s + (unsigned)((mm * BK + (km ^ swm)) * sizeof(cplx));

  int ld_stage = 0;
  auto load_tile = [&](int kl, int stage) {
    const int k0 = kl * BK;
    const unsigned so = (unsigned)(stage * STAGE_A * sizeof(cplx)), sob = (unsigned)(stage * STAGE_B * sizeof(cplx));
    if (k0 + BK <= m0) {
      const char *p = pD + k0 * ldab;
#pragma unroll
      for (int r = 0; r < RA; ++r) cp16(dD + so + (unsigned)(r * 2 * LDA_S * sizeof(cplx)), p + (2 * r) * ldab, szd);
    } else if (k0 >= m0 + BM) {
      const char *p = pM + (long long)k0 * (long long)sizeof(cplx);
      const bool kok = k0 + km < M;  // false only in a ragged last k-tile
#pragma unroll
      for (int r = 0; r < RA; ++r)
        cp16(dM + so + (unsigned)(r * MSTEP * BK * sizeof(cplx)), p + (MSTEP * r) * ldab, kok ? szm[r] : 0u);
    } else {  // the diagonal block: per element
#pragma unroll
      for (int r = 0; r < RA; ++r) {
        const int row = m0 + md, col = k0 + kd + 2 * r;
        const bool ok = row < M && col < M;
        const cplx *src = col > row ? A + (size_t)col + (size_t)row * g.lda : A + (size_t)row + (size_t)col * g.lda;
        cp16(dD + so + (unsigned)(r * 2 * LDA_S * sizeof(cplx)), ok ? src : A, ok ? 16u : 0u);
      }
    }
#pragma unroll
    for (int r = 0; r < RB; ++r)
      cp16(dB + sob + (unsigned)(r * MSTEP * BK * sizeof(cplx)), pB + (long long)k0 * (long long)sizeof(cplx) + (long long)(r * MSTEP) * ldbb, k0 + km < M ? 16u : 0u);
  };

  double c1[2][2][2], c2[2][2][2], c3[2][2][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) c1[i][j][0] = c1[i][j][1] = c2[i][j][0] = c2[i][j][1] = c3[i][j][0] = c3[i][j][1] = 0.0;

  // Order of the k-tiles: by blocks of 64 columns, block J = (r - I) mod tiles_m in round r (I = this CTA's block row).
  // The lower-triangle block {I, J} is needed by the CTAs I and J only, and this order has both of them read it in the
  // same round r, so the second reader finds it in L2 (the CTAs of one matrix are launched together and do the same
  // work per round); with J = 0, 1, 2, ... the two readers are |I - J| rounds apart and both go to DRAM.
  const int I = m0 / BM;
  auto block_of = [&](int r) { int J = r - I; return J < 0 ? J + tiles_m : J; };
  int ld_r = 0, ld_kt = block_of(0) * (BM / BK), ld_end = min(ld_kt + BM / BK, nkt);
  auto load_next = [&]() {  // loads the next k-tile of the sequence into the stage of its sequence number
    if (ld_r < tiles_m) load_tile(ld_kt, ld_stage);
    ld_stage = ld_stage + 1 == ST ? 0 : ld_stage + 1;
    if (++ld_kt >= ld_end) {
      ++ld_r;
      ld_kt = block_of(ld_r) * (BM / BK);
      ld_end = min(ld_kt + BM / BK, nkt);
    }
  };
#pragma unroll
  for (int s = 0; s < ST - 1; ++s) {
    load_next();
    cp_commit();
  }
  const int sw = (gq & 1) << 2;
  const cplx *fa0 = As + tq * LDA_S + warp * 16 + gq, *fat0 = As + (warp * 16 + gq) * BK + tq, *fb0 = Bs + gq * BK + tq;
  int stage = 0;
  // MODE 0: left of the diagonal block, 1: right of it (every element conjugated), 2: inside it
  auto k_tile = [&](int kt, auto mode) {
    constexpr int MODE = decltype(mode)::value;
    cp_wait<ST - 2>();
    __syncthreads();
    load_next();
    cp_commit();
    const cplx *fa = (MODE == 1 ? fat0 : fa0) + stage * STAGE_A, *fb = fb0 + stage * STAGE_B;
    stage = stage + 1 == ST ? 0 : stage + 1;
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      cplx a[2], b[2];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi) a[mi] = MODE == 1 ? fa[mi * 8 * BK + (kk ^ sw)] : fa[kk * LDA_S + mi * 8];
#pragma unroll
      for (int ni = 0; ni < 2; ++ni) b[ni] = fb[ni * 8 * BK + (kk ^ sw)];
      if (MODE == 1) {
#pragma unroll
        for (int mi = 0; mi < 2; ++mi) a[mi].y = __hiloint2double(__double2hiint(a[mi].y) ^ (int)0x80000000, __double2loint(a[mi].y));
      } else if (MODE == 2) {
#pragma unroll
        for (int mi = 0; mi < 2; ++mi) {
          const int mg = m0 + warp * 16 + mi * 8 + gq, kg = kt * BK + kk + tq;
          int hi = __double2hiint(a[mi].y), lo = __double2loint(a[mi].y);
          hi = kg > mg ? hi ^ (int)0x80000000 : hi;
          hi = kg == mg ? 0 : hi;
          lo = kg == mg ? 0 : lo;
          a[mi].y = __hiloint2double(hi, lo);
        }
      }
      double bs[2];
#pragma unroll
      for (int ni = 0; ni < 2; ++ni) bs[ni] = b[ni].x + b[ni].y;
#pragma unroll
      for (int mi = 0; mi < 2; ++mi) {
        const double as = a[mi].x + a[mi].y;
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) dmma(c1[mi][ni][0], c1[mi][ni][1], a[mi].x, b[ni].x);
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) dmma(c2[mi][ni][0], c2[mi][ni][1], a[mi].y, b[ni].y);
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) dmma(c3[mi][ni][0], c3[mi][ni][1], as, bs[ni]);
      }
    }
  };
  for (int r = 0; r < tiles_m; ++r) {
    const int J = block_of(r), kt0 = J * (BM / BK), kt1 = min(kt0 + BM / BK, nkt);
    if (J < I) {
      for (int kt = kt0; kt < kt1; ++kt) k_tile(kt, std::integral_constant<int, 0>());
    } else if (J > I) {
      for (int kt = kt0; kt < kt1; ++kt) k_tile(kt, std::integral_constant<int, 1>());
    } else {
      for (int kt = kt0; kt < kt1; ++kt) k_tile(kt, std::integral_constant<int, 2>());
    }
  }
  cp_wait<0>();

  const bool has_beta = (g.beta.x != 0.0 || g.beta.y != 0.0);
#pragma unroll
  for (int mi = 0; mi < 2; ++mi) {
    const int row = m0 + warp * 16 + mi * 8 + gq;
    if (row >= M) continue;
#pragma unroll
    for (int ni = 0; ni < 2; ++ni) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int col = ni * 8 + tq * 2 + j;
        const double t1 = c1[mi][ni][j], t2 = c2[mi][ni][j];
        cplx v = cmul(g.alpha, cmake(t1 - t2, c3[mi][ni][j] - t1 - t2));
        cplx *dst = C + (size_t)row + (size_t)col * g.ldc;
        if (has_beta) v = cadd(v, cmul(g.beta, *dst));
        *dst = v;
      }
    }
  }
}
void launch_hemm16(const GemmDesc &g, cudaStream_t s) {
  constexpr int CPS = 4;
  constexpr size_t smem = (size_t)4 * (8 * (64 + 2) + 16 * 8) * sizeof(cplx);
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(hemm16_kernel<CPS, 8, 4>, (int)smem, attr_mask);
  const int tm = (g.M + 63) / 64;
  hemm16_kernel<CPS, 8, 4><<<tm * g.ncells * g.inner, 128, smem, s>>>(g);
}

template <int OPA, int OPB, int HERM, int BM = 32, int BN = 32, int NT = 128, int MI = 2, int BK = 8, int STAGES = 4, int CPS = 640 / NT>
void launch_one(const GemmDesc &g, cudaStream_t s) {
  constexpr size_t smem = smem_bytes<BM, BN, BK, STAGES>();
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(zgemm_kernel<OPA, OPB, HERM, BM, BN, NT, MI, BK, STAGES, CPS>, (int)smem, attr_mask);
  const int tm = (g.M + BM - 1) / BM, zz = g.ncells * g.inner * (g.ksplit > 1 ? g.ksplit : 1);
  dim3 grid(tm * zz, (g.N + BN - 1) / BN, 1);
  if (g.flags & BS_GEMM_LOWER_ONLY) grid = dim3((BM / BN) * (tm * (tm + 1) / 2) * zz, 1, 1);  // requires M == N
  zgemm_kernel<OPA, OPB, HERM, BM, BN, NT, MI, BK, STAGES, CPS><<<grid, NT, smem, s>>>(g);
}
}  // namespace

void launch_zgemm(const GemmDesc &g, cudaStream_t s) {
  if (g.M <= 0 || g.N <= 0 || g.ncells * g.inner <= 0) return;
  double work = 8.0 * g.K * (double)g.ncells * g.inner;
  work *= (g.flags & BS_GEMM_LOWER_ONLY) ? 0.5 * g.M * (g.M + 1.0) : (double)g.M * g.N;
  if (g.flags & (BS_GEMM_KLO_ROW | BS_GEMM_KHI_ROW | BS_GEMM_KLO_COL | BS_GEMM_KHI_COL)) work *= 0.5;
  KScope ks(g.kclass ? g.kclass : KC_OTHER, work, s);
  // C aliasing A (the panel solve of the Cholesky factorisation, A21 <- A21 inv(L11)^H): a CTA must own complete rows,
  // i.e. one column tile only; 16 x 64 tiles (1 x 4 warps) serve N <= 64
  if (g.C.bases == g.A.bases && g.C.single == g.A.single && g.C.off == g.A.off && g.opA == 0 && g.opB == 1 &&
      g.N <= 64 && g.flags == 0) {
    launch_one<0, 1, 0, 16, 64>(g, s);
    return;
  }
  if (g.N == 16 && g.opA == 0 && g.opB == 0 && g.flags == BS_GEMM_A_HERM_LOWER && g.ksplit <= 1) {
    launch_hemm16(g, s);
    return;
  }
  if (g.N <= 16 && g.opA == 0 && g.opB == 0 && !(g.flags & BS_GEMM_LOWER_ONLY)) {  // band width 16: 64 x 16 tiles
    if (g.flags & BS_GEMM_A_HERM_LOWER) launch_one<0, 0, 1, 64, 16>(g, s);
    else launch_one<0, 0, 0, 64, 16>(g, s);
    return;
  }
  if (g.flags & BS_GEMM_A_HERM_LOWER) { launch_one<0, 0, 1>(g, s); return; }  // requires opA == opB == 0, K == M
  if (g.opA == 0 && g.opB == 0) launch_one<0, 0, 0>(g, s);
  else if (g.opA == 0 && g.opB == 1) launch_one<0, 1, 0>(g, s);
  else if (g.opA == 1 && g.opB == 0 && g.M <= 48 && g.M % 32 != 0 && g.flags == 0) launch_one<1, 0, 0, 16, 32, 64>(g, s);  // Gram products of the band reduction (M = 16, 48): 16-row tiles waste no half tile
  else if (g.opA == 1 && g.opB == 0) launch_one<1, 0, 0>(g, s);
  else launch_one<1, 1, 0>(g, s);
}

}  // namespace bsk
