// S6, stage 2: Hermitian band (width B, lower storage with bulge space, ldab = 2B) -> real symmetric tridiagonal by
// Householder bulge chasing (column-wise elimination, Schwarz / Lang).  DESIGN.md section 5 (S6, stage 2).
//
// Sweep i annihilates column i below the sub-diagonal and chases the bulge down the band in steps of B columns.  Step k
// of sweep i works on the window of B storage columns [J, J + B), J = i + 1 + k B (rows J .. J + 2B - 1):
//   D = A[J:J+L, J:J+L]  (Hermitian diagonal block)    D <- H^H D H        p = tau D v, w = p - tau/2 (p^H v) v,
//                                                                          D -= v w^H + w v^H
//   C = A[J+L:J+L+L2, J:J+L]  (block below it)         u = C v, x = C[:,0] - tau u, (v2, tau2) = larfg(x),
//                                                      C <- H2^H (C H):  C -= (tau u) v^H + v2 y^H,
//                                                      y = tau2 (v2^H C - (v2^H tau u) v^H)^H,  C[:,0] = beta2 e_1
// The D half and the C half of a step do not depend on each other (only v, tau come in; v2, tau2 go out), so a team
// runs them on different warps at the same time: NW "D warps" and NW "C warps" per team (NW = 2 for B = 32, else 1).
// Every warp keeps its tiles of the block in REGISTERS in the accumulator layout of mma.sync.m8n8k4.f64 (lane (g, t),
// g = lane / 4, t = lane % 4, holds row 8 rt + g, columns 8 ct + 2 t + {0, 1} of tile (rt, ct)): the two matrix-vector
// products are DFMA row / column sums over the register tiles, and each complex rank-2 update
//   X -= a b^H + c d^H    is exactly ONE real DMMA of depth 4 per 8 x 8 tile for the real part and one for the imaginary:
//   Re: [a_re a_im c_re c_im] [b_re; b_im; d_re; d_im],   Im: [a_im -a_re c_im -c_re] [same]
// (8 x fewer issued instructions than the DFMA form; the chase is bound by instruction issue and latency, not by flops).
//
// Sweep i+1 may run two steps behind sweep i (their windows are then disjoint storage columns).  G teams run G
// consecutive sweeps ("a train") in lock step, one macro-step = one step of every team + one CTA barrier, on a ring of
// Wc band columns in shared memory: element (r, c), c <= r <= c + 2B - 1, lives at ring[(c mod Wc) * 2B + (r - c)].
// Small n: the whole band is loaded once and the teams run one continuous pipeline over all sweeps (one CTA per matrix).
// Large n: the band streams through the ring; NIO I/O warps write back the columns the train has left behind and fetch
// the ones its leading sweep needs next, under the arithmetic.  Trains are TASKS handed out by an atomic counter in
// train-major order over a group of matrices, so every SM is busy whatever the batch size and several CTAs may work on
// consecutive trains of one matrix at the same time, each following its predecessor through L2: train T publishes
// "columns < X are final and written back" in progress[m][T] (release), train T+1 waits for it (acquire) before it
// fetches them.  DESIGN.md section 5 states the ring-slot lifetime argument and the measured cost of close followers.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int NIO = 2;  // I/O warps of the streamed variant (four left room for six teams of two warps; two for seven: C5 35.8 -> 34.5 ms, C3 6.29 -> 6.06)

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ cplx shfl_c(cplx v, int src) {
  return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
__device__ __forceinline__ double warp_sum(double x) {  // butterfly: every lane gets the same bits
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}
__device__ __forceinline__ cplx shfl_xor_c(cplx v, int m) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}
// Transposed reduction of NV values per lane over a group of lanes (stride s, 2s, ...): at every stage a lane keeps
// half of its values and receives the partner's partial sums of those, so the stages move NV/2, NV/4, ... values instead
// of NV each, and the lane ends with the total of ONE value (index returned in `own`); when a single value is left the
// remaining stages are plain butterflies.  A kept sum is own + partner, exactly what the butterfly `x += shfl_xor(x)`
// forms in that lane, and a + b = b + a bit for bit: the totals are the butterfly's bits.
template <int NV, int STAGES>
__device__ __forceinline__ cplx reduce_transposed(cplx (&v)[NV], int bits, int stride, int &own) {
  static_assert(NV == 1 || NV == 2 || NV == 4, "");
  own = 0;
  cplx a;
  int st = 0;
  if (NV == 4) {
    const int b0 = bits & 1;
    const cplx k0 = b0 ? v[1] : v[0], k1 = b0 ? v[3] : v[2], s0 = b0 ? v[0] : v[1], s1 = b0 ? v[2] : v[3];
    v[0] = cadd(k0, shfl_xor_c(s0, stride));
    v[1] = cadd(k1, shfl_xor_c(s1, stride));
    own = b0;
    const int b1 = (bits >> 1) & 1;
    const cplx k = b1 ? v[1] : v[0], sd = b1 ? v[0] : v[1];
    a = cadd(k, shfl_xor_c(sd, 2 * stride));
    own += 2 * b1;
    st = 2;
  } else if (NV == 2) {
    const int b0 = bits & 1;
    const cplx k = b0 ? v[1] : v[0], sd = b0 ? v[0] : v[1];
    a = cadd(k, shfl_xor_c(sd, stride));
    own = b0;
    st = 1;
  } else {
    a = v[0];
  }
#pragma unroll
  for (; st < STAGES; ++st) a = cadd(a, shfl_xor_c(a, stride << st));
  return a;
}
__device__ __forceinline__ void named_bar(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}

template <int B, int NW>
struct Cfg {
  static constexpr int LD = 2 * B, TR = B / 8, TC = B / 8, TCW = TC / NW;
  static constexpr int TW = 2 * NW;        // warps per team
  static constexpr int TT = 32 * TW;       // threads per team
  static constexpr int MAXT = NW >= 4 ? 896 : 512;  // threads per CTA the kernels are compiled for
  // team scratch (complex elements): v (two parities), tau (two parities, padded), w, tau u, y, C[:,0], partial p, partial u
  static constexpr int O_V = 0, O_TAU = 2 * B, O_W = 2 * B + 4, O_TU = O_W + B, O_Y = O_TU + B, O_C0 = O_Y + B,
                       O_P = O_C0 + B, O_U = O_P + NW * B, SCR = O_U + NW * B;
  static_assert(TC % NW == 0, "tile columns split over the role's warps");
};

// Complex products and sums of products with EXPLICIT fused multiply-adds: this file is compiled without implicit contraction
// (so that the copies of a step inlined into different kernels round identically); explicit fma() calls are DFMAs in every
// copy, one instruction and one rounding instead of a DMUL and a DADD.
__device__ __forceinline__ cplx cmul_f(cplx a, cplx b) {
  return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ cplx cmulc_f(cplx a, cplx b) {  // a * conj(b)
  return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -(a.x * b.y)));
}
__device__ __forceinline__ double sumsq_f(double a, double b) { return fma(a, a, b * b); }

// The norm of a reflector's vector and its reciprocal, and a reciprocal, without the IEEE square root and division: their
// fix-up sequences are ~25 dependent instructions each on the chain of every step.  rsqrt is good to 1 ulp, the Newton
// step makes s * rsqrt(s) a square root good to about 1 ulp, the two Newton steps on rcp.approx (2^-23) a reciprocal
// good to about 1 ulp: H = I - tau v v^H stays unitary to a few ulp (tau, v and beta are formed from the same values),
// which is all the backward stability of the chase needs.  The subnormal range is flushed (d < 2.3e-308).
__device__ __forceinline__ void norm_and_inverse(double s, double &nrm, double &inv) {
  inv = rsqrt(s);
  nrm = s * inv;
  nrm = fma(fma(-nrm, nrm, s), 0.5 * inv, nrm);
}
__device__ __forceinline__ double fast_rcp(double d) {
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;\n" : "=d"(x) : "d"(d));
  double e = fma(-d, x, 1.0);
  x = fma(x, e, x);
  e = fma(-d, x, 1.0);
  return fma(x, e, x);
}

// LAPACK zlarfg on a vector spread over the 32 lanes of a warp (x valid for l < len; other lanes must hold 0):
// H = I - tau v v^H, H^H x = beta e_1, beta real, v[0] = 1.  Returns v in x.
__device__ __forceinline__ void warp_larfg(cplx &x, int len, int l, cplx &tau, double &beta) {
  const double ss = warp_sum((l >= 1 && l < len) ? sumsq_f(x.x, x.y) : 0.0);
  const cplx al = shfl_c(x, 0);
  if (ss == 0.0 && al.y == 0.0) {
    tau = cmake(0.0, 0.0);
    beta = al.x;
    x = (l == 0) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
    return;
  }
  double nrm, inrm;
  norm_and_inverse(sumsq_f(al.x, al.y) + ss, nrm, inrm);
  beta = -copysign(nrm, al.x);
  const double ib = -copysign(inrm, al.x);
  tau = cmake((beta - al.x) * ib, -al.y * ib);
  const double dr = al.x - beta, di = al.y, den = fast_rcp(sumsq_f(dr, di));
  const cplx scale = cmake(dr * den, -di * den);
  if (l == 0) x = cmake(1.0, 0.0);
  else if (l < len) x = cmul_f(x, scale);
  else x = cmake(0.0, 0.0);
}

// Fragment sources of a rank-2 update X -= a b^H + c d^H (vectors stored as interleaved complex in shared memory):
// A fragments of tile row R (lane (g, t) holds depth t of row g):  Re: -[a_re a_im c_re c_im][t],  Im: [-a_im a_re -c_im c_re][t]
// B fragment of tile column Cc (lane holds depth t of column g):        [b_re b_im d_re d_im][t]
__device__ __forceinline__ void frag_rows(const cplx *a, const cplx *c, int idx, int t, double &fre, double &fim) {
  const double *vec = reinterpret_cast<const double *>(t < 2 ? a : c) + 2 * idx;
  const double same = vec[t & 1], other = vec[(t & 1) ^ 1];
  fre = -same;
  fim = (t & 1) ? other : -other;
}
__device__ __forceinline__ double frag_cols(const cplx *b, const cplx *d, int idx, int t) {
  return (reinterpret_cast<const double *>(t < 2 ? b : d) + 2 * idx)[t & 1];
}

// ---------------------------------------------------------------------------------------------- the D half of a step
// D <- H^H D H on the L x L Hermitian block at (J, J); v, tau of the step are in the team scratch.  Warp rw of the NW
// D warps owns the tile columns ctg(rw, .) (all tile rows); tiles strictly above the diagonal are only read.
// FULL: the block is complete (L = B): every mask below is true and is compiled out (team-uniform choice, same bits).
template <int B, int NW, bool FULL>
__device__ __forceinline__ void step_D(cplx *ring, int Wc, int sJ, cplx *ts, const cplx *vb, cplx tau, int L, int rw_,
                                       int lane, int bar_id) {
  const int rw = NW == 1 ? 0 : rw_;  // (one warp per half: a compile-time zero, the tile positions below become constants)
  using C = Cfg<B, NW>;
  constexpr int LD = C::LD, TR = C::TR, TCW = C::TCW;
  const int g = lane >> 2, t = lane & 3;
  auto ctg = [&](int ci) { return (NW == 2 && TCW == 2) ? (ci == 0 ? rw : C::TC - 1 - rw) : rw * TCW + ci; };
  double tre[TR][TCW][2], tim[TR][TCW][2];
  // Ring addresses are formed as (column base - column) + row and (row base - row) + column, never as
  // base + (row - column): nvcc 12.9 turns the latter into `base | (row - column)` inside the branch where the
  // difference is known to be non-negative and then reuses that value, + 8, for the neighbouring tile, where it is not.
  int rs[TR];  // (ring offset of storage column J + r) - r for this lane's rows: the mirrored upper part
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) {
    int sl = sJ + 8 * rt + g;
    sl -= sl >= Wc ? Wc : 0;
    rs[rt] = sl * LD - (8 * rt + g);
  }
  cplx vc[TCW][2];
  cplx acc[TR];
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) acc[rt] = cmake(0.0, 0.0);
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int c = 8 * ctg(ci) + 2 * t + j;
      int sl = sJ + c;
      sl -= sl >= Wc ? Wc : 0;
      const int cs = sl * LD - c;
      vc[ci][j] = vb[c];
#pragma unroll
      for (int rt = 0; rt < TR; ++rt) {
        const int r = 8 * rt + g;
        const bool low = r >= c;
        const cplx a = ring[low ? cs + r : rs[rt] + c];  // lower part as stored, upper part mirrored
        const bool ok = FULL || (r < L && c < L);
        tre[rt][ci][j] = ok ? a.x : 0.0;
        tim[rt][ci][j] = (ok && r != c) ? (low ? a.y : -a.y) : 0.0;
      }
    }
  }
  // p = D v: partial row sums over this warp's columns, then over the four lanes of a row (transposed reduction: lane
  // (g, t), t < TR, ends with the sum of row 8 t + g)
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) {
#pragma unroll
    for (int ci = 0; ci < TCW; ++ci)
#pragma unroll
      for (int j = 0; j < 2; ++j) cfma(acc[rt], cmake(tre[rt][ci][j], tim[rt][ci][j]), vc[ci][j]);
  }
  {
    int own;
    const cplx a = reduce_transposed<TR, 2>(acc, t, 1, own);
    if (t < TR) ts[C::O_P + rw * B + 8 * own + g] = a;
  }
  if (NW > 1) named_bar(bar_id, 32 * NW);
  else __syncwarp();
  // lane l = row l: p = tau D v, w = p - tau/2 (p^H v) v   (every D warp computes the same bits).  For B < 32 the upper
  // lanes mirror the lower ones, so the lane sums need log2(B) butterfly stages.
  const int l = B < 32 ? (lane & (B - 1)) : lane;
  cplx p = ts[C::O_P + l];
#pragma unroll
  for (int w2 = 1; w2 < NW; ++w2) p = cadd(p, ts[C::O_P + w2 * B + l]);
  p = cmul_f(tau, p);
  const cplx v = vb[l];
  const bool in = FULL || l < L;
  double sr = in ? fma(p.x, v.x, p.y * v.y) : 0.0, si = in ? fma(p.x, v.y, -(p.y * v.x)) : 0.0;  // p^H v
#pragma unroll
  for (int o = (B < 32 ? B : 32) / 2; o > 0; o >>= 1) {
    sr += __shfl_xor_sync(0xffffffffu, sr, o);
    si += __shfl_xor_sync(0xffffffffu, si, o);
  }
  const cplx alpha = cmul_f(cmake(-0.5 * tau.x, -0.5 * tau.y), cmake(sr, si));
  cplx w = p;
  cfma(w, alpha, v);
  if (lane < B) ts[C::O_W + lane] = in ? w : cmake(0.0, 0.0);
  __syncwarp();
  // D -= v w^H + w v^H  (a, b, c, d) = (v, w, w, v)
  const cplx *wv = ts + C::O_W;
  double are[TR], aim[TR];
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) frag_rows(vb, wv, 8 * rt + g, t, are[rt], aim[rt]);
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
    const int ct = ctg(ci);
    const double bf = frag_cols(wv, vb, 8 * ct + g, t);
#pragma unroll
    for (int rt = 0; rt < TR; ++rt) {
      if (rt >= ct) {  // (warp-uniform) tiles above the diagonal are never stored
        dmma884(tre[rt][ci][0], tre[rt][ci][1], are[rt], bf);
        dmma884(tim[rt][ci][0], tim[rt][ci][1], aim[rt], bf);
      }
    }
  }
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int c = 8 * ctg(ci) + 2 * t + j;
      int sl = sJ + c;
      sl -= sl >= Wc ? Wc : 0;
      const int cs = sl * LD - c;
#pragma unroll
      for (int rt = 0; rt < TR; ++rt) {
        const int r = 8 * rt + g;
        if (r >= c && (FULL || r < L)) ring[cs + r] = cmake(tre[rt][ci][j], r == c ? 0.0 : tim[rt][ci][j]);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- the C half of a step
// C <- H2^H (C H) on the L2 x L block below D; produces the next reflector (v2 -> vnext, tau2 -> *tau_next).  Warp rw of
// the NW C warps owns the tile columns rw TCW .. (rw + 1) TCW - 1 (all tile rows).
// FULL: both blocks are complete (L = L2 = B): the masks are compiled out.
template <int B, int NW, bool FULL>
__device__ __forceinline__ void step_C(cplx *ring, int Wc, int sJ, cplx *ts, const cplx *vb, cplx *vnext, cplx *tau_next,
                                       cplx tau, int L, int L2, int rw_, int lane, int bar_id, int team_bar) {
  const int rw = NW == 1 ? 0 : rw_;
  using C = Cfg<B, NW>;
  constexpr int LD = C::LD, TR = C::TR, TCW = C::TCW;
  const int g = lane >> 2, t = lane & 3;
  double tre[TR][TCW][2], tim[TR][TCW][2];
  cplx vc[TCW][2];
  cplx acc[TR];
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) acc[rt] = cmake(0.0, 0.0);
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int c = 8 * (rw * TCW + ci) + 2 * t + j;
      int sl = sJ + c;
      sl -= sl >= Wc ? Wc : 0;
      const int cs = sl * LD + ((FULL || c < L) ? L - c : 0);  // (a masked column reads its own first entries)
      vc[ci][j] = vb[c];
#pragma unroll
      for (int rt = 0; rt < TR; ++rt) {
        const int r = 8 * rt + g;
        cplx a = ring[cs + r];
        const bool ok = FULL || (r < L2 && c < L);
        tre[rt][ci][j] = ok ? a.x : 0.0;
        tim[rt][ci][j] = ok ? a.y : 0.0;
      }
    }
  }
  // u = C v: partial row sums (transposed reduction over the four lanes of a row); C[:,0] goes along
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) {
#pragma unroll
    for (int ci = 0; ci < TCW; ++ci)
#pragma unroll
      for (int j = 0; j < 2; ++j) cfma(acc[rt], cmake(tre[rt][ci][j], tim[rt][ci][j]), vc[ci][j]);
    if (t == 0 && rw == 0) ts[C::O_C0 + 8 * rt + g] = cmake(tre[rt][0][0], tim[rt][0][0]);
  }
  asm volatile("bar.arrive %0, %1;\n" ::"r"(team_bar), "r"(C::TT) : "memory");  // releases the D warps of the team
  {
    int own;
    const cplx a = reduce_transposed<TR, 2>(acc, t, 1, own);
    if (t < TR) ts[C::O_U + rw * B + 8 * own + g] = a;
  }
  if (NW > 1) named_bar(bar_id, 32 * NW);
  else __syncwarp();
  // lane l = row l of C: x = C[:,0] - tau u (conj(v[0]) = 1), then the reflector that annihilates x below its first entry.
  // zlarfg, branch-free: no reflector when the block has a single row (L2 <= 1) or x is already e_1-shaped.
  // For B < 32 the upper lanes mirror the lower ones, so the lane sums need log2(B) butterfly stages.
  const int l = B < 32 ? (lane & (B - 1)) : lane;
  cplx u = ts[C::O_U + l];
#pragma unroll
  for (int w2 = 1; w2 < NW; ++w2) u = cadd(u, ts[C::O_U + w2 * B + l]);
  const bool in = FULL || l < L2;
  cplx tu = cmul_f(tau, u);
  tu.x = in ? tu.x : 0.0;
  tu.y = in ? tu.y : 0.0;
  cplx x = csub(ts[C::O_C0 + l], tu);
  x.x = in ? x.x : 0.0;
  x.y = in ? x.y : 0.0;
  // three lane reductions in one butterfly: |x[1:]|^2 and sum_{l>=1} conj(x_l) (tau u)_l, which gives
  // s = v2^H (tau u) = (tau u)_0 + conj(scale) sum_{l>=1} conj(x_l) (tau u)_l  without a second pass over the lanes
  double ss = l >= 1 ? sumsq_f(x.x, x.y) : 0.0;
  double sdr = l >= 1 ? fma(x.x, tu.x, x.y * tu.y) : 0.0;
  double sdi = l >= 1 ? fma(x.x, tu.y, -(x.y * tu.x)) : 0.0;
#pragma unroll
  for (int o = (B < 32 ? B : 32) / 2; o > 0; o >>= 1) {
    ss += __shfl_xor_sync(0xffffffffu, ss, o);
    sdr += __shfl_xor_sync(0xffffffffu, sdr, o);
    sdi += __shfl_xor_sync(0xffffffffu, sdi, o);
  }
  const cplx al = shfl_c(x, 0), tu0 = shfl_c(tu, 0);
  const bool norefl = L2 <= 1, trivial = norefl || (ss == 0.0 && al.y == 0.0);
  double nrm, inrm;
  norm_and_inverse(sumsq_f(al.x, al.y) + ss, nrm, inrm);
  const double beta2 = trivial ? 1.0 : -copysign(nrm, al.x);
  const double ib = trivial ? 1.0 : -copysign(inrm, al.x);
  cplx tau2 = cmake((beta2 - al.x) * ib, -al.y * ib);
  tau2.x = trivial ? 0.0 : tau2.x;
  tau2.y = trivial ? 0.0 : tau2.y;
  const double dr = al.x - beta2, di = al.y;
  const double den = fast_rcp(sumsq_f(dr, di));
  cplx scale = cmake(dr * den, -di * den);
  scale.x = trivial ? 0.0 : scale.x;
  scale.y = trivial ? 0.0 : scale.y;
  cplx v2 = cmul_f(x, scale);
  v2.x = l == 0 ? 1.0 : v2.x;
  v2.y = l == 0 ? 0.0 : v2.y;
  const cplx sv = cadd(tu0, cmulc_f(cmake(sdr, sdi), scale));  // (tau u)_0 + conj(scale) sum conj(x_l) (tau u)_l
  const double s_re = sv.x, s_im = sv.y;
  if (lane < B) {
    ts[C::O_TU + lane] = tu;
    vnext[lane] = v2;
  }
  if (lane == 0) *tau_next = tau2;
  __syncwarp();
  // z0 = v2^H C over this warp's columns: column sums over the tile rows, then over the eight lanes of a column by a
  // transposed reduction: lane (g, t), g < 2 TCW, ends with the sum of column 8 (rw TCW + g / 2) + 2 t + g % 2 and forms
  // that column's entry of y alone
  cplx z[2 * TCW];
#pragma unroll
  for (int q = 0; q < 2 * TCW; ++q) z[q] = cmake(0.0, 0.0);
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) {
    const cplx vr = vnext[8 * rt + g];
#pragma unroll
    for (int ci = 0; ci < TCW; ++ci)
#pragma unroll
      for (int j = 0; j < 2; ++j) cfmac(z[2 * ci + j], vr, cmake(tre[rt][ci][j], tim[rt][ci][j]));
  }
  {
    int own;
    const cplx zs = reduce_transposed<2 * TCW, 3>(z, g, 4, own);
    const int co = 8 * (rw * TCW + (own >> 1)) + 2 * t + (own & 1);
    // y = tau2 conj(z0 - s conj(v)) = tau2 (conj(z0) - conj(s) v)
    const cplx vcj = vb[co];
    const cplx q = cmake(zs.x - fma(s_re, vcj.x, s_im * vcj.y), -zs.y - fma(s_re, vcj.y, -(s_im * vcj.x)));
    if (g < 2 * TCW) ts[C::O_Y + co] = cmul_f(tau2, q);
  }
  __syncwarp();
  // C -= (tau u) v^H + v2 y^H   (a, b, c, d) = (tau u, v, v2, y)
  const cplx *tuv = ts + C::O_TU, *yv = ts + C::O_Y;
  double are[TR], aim[TR];
#pragma unroll
  for (int rt = 0; rt < TR; ++rt) frag_rows(tuv, vnext, 8 * rt + g, t, are[rt], aim[rt]);
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
    const double bf = frag_cols(vb, yv, 8 * (rw * TCW + ci) + g, t);
#pragma unroll
    for (int rt = 0; rt < TR; ++rt) {
      dmma884(tre[rt][ci][0], tre[rt][ci][1], are[rt], bf);
      dmma884(tim[rt][ci][0], tim[rt][ci][1], aim[rt], bf);
    }
  }
  // the annihilated column: C[:,0] = beta2 e_1 exactly (x itself when no reflector was formed)
  if (rw == 0 && t == 0) {
    const cplx c00 = norefl ? al : cmake(trivial ? al.x : beta2, 0.0);
#pragma unroll
    for (int rt = 0; rt < TR; ++rt) {
      const bool first = rt == 0 && g == 0;
      tre[rt][0][0] = first ? c00.x : 0.0;
      tim[rt][0][0] = first ? c00.y : 0.0;
    }
  }
#pragma unroll
  for (int ci = 0; ci < TCW; ++ci) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int c = 8 * (rw * TCW + ci) + 2 * t + j;
      int sl = sJ + c;
      sl -= sl >= Wc ? Wc : 0;
      const int cs = sl * LD + (L - c);
#pragma unroll
      for (int rt = 0; rt < TR; ++rt) {
        const int r = 8 * rt + g;
        if (FULL || (r < L2 && c < L)) ring[cs + r] = cmake(tre[rt][ci][j], tim[rt][ci][j]);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- one step of one sweep
// Executed by all 2 NW warps of a team (role 0 = D warps, 1 = C warps).  State (i, k, J, L, finished) is identical in
// every thread of the team.  Named barriers: 1 + team (whole team, only at k = 0), 5 + team / 9 + team (the D / C pair
// of a B = 32 team; G <= 4 there), 15 (I/O warps).
// The head of sweep i: the reflector that annihilates column i below the sub-diagonal (into the parity-0 buffers of the team
// scratch); d[i], e[i] are final.  One warp.  Column i is final once sweep i - 1 has finished its step 0, i.e. one macro-step
// before sweep i may start: a team that is idle then computes the head there (`head_done`), beside the steps of the
// other teams, instead of at the start of its own step 0, where every second macro-step of the pipeline would wait for it.
template <int B, int NW>
__device__ __forceinline__ void sweep_head(const cplx *ring, int Wc, cplx *ts, int n, int i, int lane, double *dg, double *eg) {
  using C = Cfg<B, NW>;
  const int L = min(B, n - 1 - i);
  const cplx *ci = ring + (size_t)(i % Wc) * C::LD;
  cplx x = lane < L ? ci[1 + lane] : cmake(0.0, 0.0);
  cplx tau0;
  double beta;
  warp_larfg(x, L, lane, tau0, beta);
  if (lane < B) ts[C::O_V + lane] = x;
  if (lane == 0) {
    ts[C::O_TAU] = tau0;
    eg[i] = beta;
    dg[i] = ci[0].x;
  }
}

template <int B, int NW>
__device__ __forceinline__ void team_step(cplx *ring, int Wc, cplx *ts, int n, int i, int &k, int &J, int &sJ, int &L,
                                          bool &finished, int role, int rw, int lane, int team, double *dg, double *eg,
                                          bool &head_done) {
  using C = Cfg<B, NW>;
  const int par = k & 1;
  cplx *vb = ts + C::O_V + par * B, *vnext = ts + C::O_V + (par ^ 1) * B;
  if (k == 0) {
    L = min(B, n - 1 - i);
    if (!head_done) {  // (team-uniform)
      if (role == 1 && rw == 0) sweep_head<B, NW>(ring, Wc, ts, n, i, lane, dg, eg);
      named_bar(1 + team, C::TT);
    }
    head_done = false;
  }
  const cplx tau = ts[C::O_TAU + par];
  const int Jn = J + L, L2 = min(B, n - Jn);
  if (role == 0) {
    // the C warps (the longer chain of the step) load their tiles first: the D warps wait until those are in registers
    if (L2 > 0) named_bar(1 + team, C::TT);
    if (L == B) step_D<B, NW, true>(ring, Wc, sJ, ts, vb, tau, L, rw, lane, 5 + team);
    else step_D<B, NW, false>(ring, Wc, sJ, ts, vb, tau, L, rw, lane, 5 + team);
  } else if (L2 > 0) {
    if (L == B && L2 == B)
      step_C<B, NW, true>(ring, Wc, sJ, ts, vb, vnext, ts + C::O_TAU + (par ^ 1), tau, L, L2, rw, lane, 9 + team, 1 + team);
    else
      step_C<B, NW, false>(ring, Wc, sJ, ts, vb, vnext, ts + C::O_TAU + (par ^ 1), tau, L, L2, rw, lane, 9 + team, 1 + team);
  }
  if (L2 <= 0) {
    finished = true;
  } else {
    sJ += L;  // ring slot of column J, kept incrementally (L <= B < Wc)
    sJ -= sJ >= Wc ? Wc : 0;
    J = Jn; L = L2; ++k;
  }
}

// ---------------------------------------------------------------------------------------------- band resident in shared memory
// One CTA per matrix, the whole band in the ring (Wc >= n), no I/O: the G teams run one continuous pipeline.  Sweep j
// starts at macro-step start[j] = max(start[j-1] + 2, finish of sweep j-G) (two blocks behind its predecessor, and its
// team must be free).
template <int B, int NW>
__global__ void __launch_bounds__(Cfg<B, NW>::MAXT) chase_resident_kernel(int n, BatchRef AB, double *d, double *e, int G, int Wc, int inner) {
  using C = Cfg<B, NW>;
  constexpr int LD = C::LD;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *ring = reinterpret_cast<cplx *>(smem_raw);
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  const cplx *ab = batch_ptr(AB, cell, mi);
  double *dg = d + (size_t)z * n, *eg = e + (size_t)z * n;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // warps [0, G NW): the D warps of teams 0 .. G-1, then the C warps (the issue arbiter favours the higher warp index:
  // the C half is the longer chain), then the I/O warps; every scheduler hosts warps of both roles
  const int role = warp >= G * NW ? 1 : 0, wr = warp - role * G * NW, team = wr / NW, rw = wr % NW;
  cplx *ts = ring + (size_t)Wc * LD + (size_t)team * C::SCR;
  int *start = reinterpret_cast<int *>(ring + (size_t)Wc * LD + (size_t)G * C::SCR);
  for (int q = tid; q < n * LD; q += blockDim.x) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(ring + q);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(ab + q));
  }
  asm volatile("cp.async.commit_group;\n" ::);
  if (tid == 0) {
    for (int j = 0; j <= n - 2; ++j) {
      int st = j == 0 ? 0 : start[j - 1] + 2;
      if (j >= G) st = max(st, start[j - G] + (n - 1 - (j - G) + B - 1) / B);
      start[j] = st;
    }
  }
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();
  const int S = n >= 2 ? start[n - 2] + 1 : 0;  // the last sweep has a single step
  int i = 0, k = 0, J = 0, sJ = 0, L = 0, next_i = team;
  bool finished = true, head_done = false;
  for (int s = 0; s < S; ++s) {
    if (finished && next_i <= n - 2 && start[next_i] == s) {
      i = next_i; k = 0; J = i + 1; sJ = J % Wc; L = 0; finished = false;
    }
    if (!finished) {
      team_step<B, NW>(ring, Wc, ts, n, i, k, J, sJ, L, finished, role, rw, lane, team, dg, eg, head_done);
      if (finished) next_i += G;
    } else if (next_i <= n - 2 && start[next_i] == s + 1) {
      // idle now, the next sweep of this team starts at the next macro-step: its column is final, its head goes here
      if (role == 1 && rw == 0) sweep_head<B, NW>(ring, Wc, ts, n, next_i, lane, dg, eg);
      head_done = true;
    }
    __syncthreads();
  }
  if (tid == 0 && n >= 1) {
    dg[n - 1] = ring[(size_t)((n - 1) % Wc) * LD].x;
    eg[n - 1] = 0.0;
  }
}

// ---------------------------------------------------------------------------------------------- band streamed through the ring
__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int *p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}

// sync[0]: task counter; sync[1 + m * ntrains + T]: progress of train T of matrix m = "band columns < progress are final
// for this train and written back to global memory" (INT_MAX once the train is done).  Zeroed before the launch.
// Task order: groups of `group` matrices; inside a group train-major (train T of every matrix of the group, then T + 1),
// so the CTAs in flight spread over about (CTAs / group) consecutive trains of each matrix of the group.  A task only
// ever waits for its predecessor train, which was handed out earlier and is running or done: no deadlock.
template <int B, int NW>
__global__ void __launch_bounds__(Cfg<B, NW>::MAXT) chase_stream_kernel(int n, BatchRef AB, double *d, double *e, int G, int Wc,
                                                           int inner, int nmat, int group, int ntrains, int *sync) {
  using C = Cfg<B, NW>;
  constexpr int LD = C::LD;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_task;
  cplx *ring = reinterpret_cast<cplx *>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ncomp = G * C::TT;
  const bool is_io = tid >= ncomp;
  const int io_tid = tid - ncomp, io_nt = (int)blockDim.x - ncomp;
  // warps [0, G NW): the D warps of teams 0 .. G-1, then the C warps (the issue arbiter favours the higher warp index:
  // the C half is the longer chain), then the I/O warps; every scheduler hosts warps of both roles
  const int role = warp >= G * NW ? 1 : 0, wr = warp - role * G * NW, team = wr / NW, rw = wr % NW;
  cplx *ts = ring + (size_t)Wc * LD + (size_t)(is_io ? 0 : team) * C::SCR;
  const int ntasks = nmat * ntrains;

  for (;;) {
    if (tid == 0) s_task = atomicAdd(&sync[0], 1);
    __syncthreads();
    const int task = s_task;
    __syncthreads();
    if (task >= ntasks) break;
    const int gi = task / (group * ntrains), rem = task - gi * group * ntrains;
    const int gsz = min(group, nmat - gi * group);
    const int T = rem / gsz, m = gi * group + rem % gsz;
    cplx *ab = batch_ptr(AB, m / inner, m % inner);
    double *dg = d + (size_t)m * n, *eg = e + (size_t)m * n;
    const int *prev = T > 0 ? sync + 1 + (size_t)m * ntrains + (T - 1) : nullptr;
    int *mine = sync + 1 + (size_t)m * ntrains + T;
    const int t0 = T * G, nvalid = min(G, n - 1 - t0);  // sweeps t0 .. t0 + nvalid - 1

    // Thread t of nt (nt a multiple of LD) moves element t % LD of the columns c0 + t / LD + j (nt / LD): the ring slot
    // is advanced incrementally and every thread keeps several independent 16-byte transfers in flight.
    auto io_load = [&](int c0, int c1, int t, int nt) {
      const int off = t % LD, cstep = nt / LD;
      int c = c0 + t / LD;
      if (c < c1) {
        int sl = c % Wc;
        const int sstep = cstep % Wc;
        for (; c < c1; c += cstep) {
          const unsigned dst = (unsigned)__cvta_generic_to_shared(ring + (size_t)sl * LD + off);
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(ab + (size_t)c * LD + off));
          sl += sstep;
          if (sl >= Wc) sl -= Wc;
        }
      }
      asm volatile("cp.async.commit_group;\n" ::);
      asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    };
    auto io_evict = [&](int c0, int c1, int t, int nt) {
      const int off = t % LD, cstep = nt / LD;
      int c = c0 + t / LD;
      if (c < c1) {
        int sl = c % Wc;
        const int sstep = cstep % Wc;
#pragma unroll 4
        for (; c < c1; c += cstep) {
          ab[(size_t)c * LD + off] = ring[(size_t)sl * LD + off];
          sl += sstep;
          if (sl >= Wc) sl -= Wc;
        }
      }
    };

    // the head of the band for this train: columns [t0, t0 + 1 + B)
    int wlo = t0, whi = min(n, t0 + 1 + B);
    if (tid == 0 && prev)
      while (ld_acquire(prev) < whi) __nanosleep(64);
    __syncthreads();
    io_load(wlo, whi, tid, blockDim.x);
    __syncthreads();

    int i = t0 + team, k = 0, J = i + 1, sJ = J % Wc, L = 0;
    bool finished = is_io || team >= nvalid, head_done = false;
    const int nsteps0 = (n - 1 - t0 + B - 1) / B;
    const int S = nsteps0 + 2 * (nvalid - 1);
    for (int s = 0; s < S; ++s) {
      // window bookkeeping (uniform, closed form): keep = first column still needed at macro-step s or later, hi = end of
      // the columns needed at macro-step s + 1.  Team g is at step s - 2g; window starts decrease with g and a later team
      // finishes later, so keep is decided by the first team that has not started (its own column t0 + g) or else by the
      // last team; hi is decided by team 0 alone (once it has reached the end of the band, hi = n stays).
      int keep, hi = whi;
      {
        const int gu = (s + 1) >> 1, gl = nvalid - 1;
        if (gu < nvalid) {
          keep = t0 + gu;
        } else {
          const int kg = s - 2 * gl, ns = (n - 1 - (t0 + gl) + B - 1) / B;
          keep = kg < ns ? t0 + gl + 1 + kg * B : n;
        }
        if (s + 1 < nsteps0) hi = max(hi, min(n, t0 + 1 + (s + 2) * B));
      }
      keep = max(keep, wlo);
      if (is_io) {
        io_evict(max(wlo, t0 + nvalid), keep, io_tid, io_nt);  // (columns < t0 + nvalid are finished sweeps: never read again)
        // progress is published every fourth macro-step (the fence costs ~2000 cycles of the I/O warps; followers are rare
        // with one group of matrices per wave of CTAs and only start a little later)
        const bool publish = (s & 3) == 3;
        if (publish) __threadfence();
        // the columns fetched below reuse ring slots of columns written back just above, in general through another
        // thread: all slot reads (and global writes) first
        named_bar(15, io_nt);
        if (io_tid == 0) {
          if (publish) st_release(mine, keep);
          if (prev && hi > whi)
            while (ld_acquire(prev) < hi) __nanosleep(20);
        }
        named_bar(15, io_nt);
        io_load(whi, hi, io_tid, io_nt);
      }
      wlo = keep; whi = hi;
      if (!finished && s >= 2 * team) {
        team_step<B, NW>(ring, Wc, ts, n, i, k, J, sJ, L, finished, role, rw, lane, team, dg, eg, head_done);
      } else if (!finished && s == 2 * team - 1) {
        // the sweep starts at the next macro-step: its column is final (the sweep before it has finished its step 0)
        if (role == 1 && rw == 0) sweep_head<B, NW>(ring, Wc, ts, n, i, lane, dg, eg);
        head_done = true;
      }
      __syncthreads();
    }
    // the tail of the window goes back; the train is done
    io_evict(max(wlo, t0 + nvalid), whi, tid, blockDim.x);
    if (T == ntrains - 1 && tid == 0) {
      dg[n - 1] = ring[(size_t)((n - 1) % Wc) * LD].x;
      eg[n - 1] = 0.0;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) st_release(mine, 0x7fffffff);
  }
}

constexpr size_t CHASE_MAX_SMEM = 226 * 1024;
// warps per role (D, C) of a team at band width 32.  Four (28 warps per CTA, 72 registers) was measured slower than two:
// C5 95.7 vs 85.6 ms, C3 16.7 vs 14.9 ms (spills, and the exchanges then span four warps)
constexpr int NW32 = 2;
template <int B, int NW>
constexpr int chase_gmax_resident() { return NW > 1 ? (Cfg<B, NW>::MAXT / Cfg<B, NW>::TT < 4 ? Cfg<B, NW>::MAXT / Cfg<B, NW>::TT : 4) : 512 / Cfg<B, NW>::TT; }
template <int B, int NW>
constexpr int chase_gmax_stream() { return NW >= 2 ? 3 : (512 - NIO * 32) / Cfg<B, NW>::TT; }
template <int B, int NW>
constexpr bool chase_fits(int n) {  // the whole band (n columns of 2B entries) beside the team scratch and the start table
  return (size_t)(n > 2 * B + 8 ? n : 2 * B + 8) * 2 * B * sizeof(cplx) +
             (size_t)chase_gmax_resident<B, NW>() * Cfg<B, NW>::SCR * sizeof(cplx) + (size_t)n * sizeof(int) <= CHASE_MAX_SMEM;
}

int g_sm_count(int dev) {
  static int cache[64] = {0};
  if (!cache[dev & 63]) cudaDeviceGetAttribute(&cache[dev & 63], cudaDevAttrMultiProcessorCount, dev);
  return cache[dev & 63];
}

template <int B, int NW>
void launch_chase_t(int n, BatchRef AB, double *d, double *e, int nmat, int inner, bool streamed, int force_g, int *sync,
                    cudaStream_t s) {
  using C = Cfg<B, NW>;
  const size_t colbytes = (size_t)C::LD * sizeof(cplx), team_bytes = (size_t)C::SCR * sizeof(cplx);
  // algorithmic work: ~n^2/(2B) steps of 48 B^2 real flops (hemv, rank-2, C v, right- and left-apply)
  KScope ks(KC_BULGE, 24.0 * n * (double)n * B * nmat, s);
  static unsigned long long m1 = 0, m2 = 0;
  if (!(streamed && n > 2 * B + 8) && chase_fits<B, NW>(n)) {
    const int Wc = max(n, 2 * B + 8);  // never fewer than a block pair of columns: masked loads stay inside the ring
    const int G = max(1, min(chase_gmax_resident<B, NW>(), (n + 2 * B - 1) / (2 * B)));
    const size_t smem = (size_t)Wc * colbytes + G * team_bytes + (size_t)n * sizeof(int);
    ensure_dyn_smem(chase_resident_kernel<B, NW>, (int)CHASE_MAX_SMEM, m1);
    chase_resident_kernel<B, NW><<<nmat, G * C::TT, smem, s>>>(n, AB, d, e, G, Wc, inner);
    return;
  }
  int G = (int)(((CHASE_MAX_SMEM - 64) / colbytes - 8) / (2 * B));
  G = max(1, min(G, chase_gmax_stream<B, NW>()));
  while (G > 1 && (size_t)(2 * G * B + 8) * colbytes + G * team_bytes > CHASE_MAX_SMEM) --G;
  if (force_g > 0) G = min(force_g, G);
  const int Wc = 2 * G * B + 8;
  const size_t smem = (size_t)Wc * colbytes + G * team_bytes;
  const int threads = G * C::TT + NIO * 32;
  const int ntrains = (n - 1 + G - 1) / G;
  ensure_dyn_smem(chase_stream_kernel<B, NW>, (int)CHASE_MAX_SMEM, m2);  // (+ 16 bytes of static shared memory)
  int dev = 0, occ = 1;
  cudaGetDevice(&dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, chase_stream_kernel<B, NW>, threads, smem);
  const int resident = g_sm_count(dev) * max(occ, 1);
  const long long ntasks = (long long)nmat * ntrains;
  const int grid = (int)min((long long)resident, ntasks);
  // One group = as many matrices as there are CTAs (train-major inside the group): a CTA that finishes train T of one
  // matrix moves on to another matrix, and train T + 1 of the first is taken up when its predecessor is far ahead or
  // done.  Measured on C5 / C3 (ms) with about c CTAs following one another on each matrix: c = 1: 87.6 / 15.2,
  // c = 2: 87.6 / 19.2, c = 3: 91.9 / 19.2, c = 4: 100.3 / 27.1, c = 6: 112 / 35.9 -- a train cannot start before its
  // predecessor is 2G + 1 macro-steps ahead, and trains are only ~35 macro-steps long, so close followers mostly wait.
  int group = max(1, grid);
  {
    // ... unless the bands of a group do not fit L2 beside one another: then half as many matrices per group (two CTAs
    // follow one another per matrix, which costs ~1 %) keep the bands L2-resident between their trains.  C5 (120 bands of
    // 0.98 MB, 126 MB of L2): DRAM traffic of the launch 16.4 -> 1.3 GB, L2 hit rate 80 -> 87 %, 35.5 -> 35.8 ms; a third
    // (0.2 GB) costs 10 %.  The task order changes no arithmetic.
    int l2 = 0;
    cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
    const double live = (double)min((long long)nmat, (long long)grid) * n * colbytes;
    if (l2 > 0 && live > 0.6 * l2) group = max(1, grid / 2);
  }
  const int ngroups = (nmat + group - 1) / group;
  group = (nmat + ngroups - 1) / ngroups;
  cudaMemsetAsync(sync, 0, sizeof(int) * (size_t)(1 + ntasks), s);
  chase_stream_kernel<B, NW><<<grid, threads, smem, s>>>(n, AB, d, e, G, Wc, inner, nmat, group, ntrains, sync);
}
}  // namespace

bool bulge_band_resident(int n, int b) {
  return b >= 32 ? chase_fits<32, NW32>(n) : (b >= 16 ? chase_fits<16, 1>(n) : chase_fits<8, 1>(n));
}
size_t sb2st_sync_ints(int n, int nmat) { return 1 + (size_t)nmat * (size_t)(n > 1 ? n - 1 : 1); }  // G >= 1 trains per matrix

// Band -> tridiagonal for every matrix of the batch.  b must be 8, 16 or 32.  sync: sb2st_sync_ints(n, nmat) ints.
void launch_sb2st(int n, int b, BatchRef AB, double *d, double *e, int ncells, int inner, cudaStream_t s, bool streamed,
                  int force_g, int *sync) {
  const int nmat = ncells * inner;
  if (b == 8) launch_chase_t<8, 1>(n, AB, d, e, nmat, inner, streamed, force_g, sync, s);
  else if (b == 16) launch_chase_t<16, 1>(n, AB, d, e, nmat, inner, streamed, force_g, sync, s);
  else launch_chase_t<32, NW32>(n, AB, d, e, nmat, inner, streamed, force_g, sync, s);
}

}  // namespace bsk
