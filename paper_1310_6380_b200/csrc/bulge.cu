// S6, stage 2: Hermitian band (width B, lower storage with bulge space, ldab = 2B) -> real symmetric tridiagonal by
// Householder bulge chasing (column-wise elimination, Schwarz / Lang).  DESIGN.md section 5 (S6, stage 2).
//
// One CTA per matrix.  Sweep i annihilates column i below the sub-diagonal and chases the bulge down the band in steps
// of B columns; step k of sweep i touches columns [i+1+kB, i+1+(k+1)B) only, so sweep i+1 can run two steps behind sweep i.
// A "train" of G consecutive sweeps is executed by G teams of NQ*B threads in lock step (team g does step s-2g at
// macro-step s) on a window of the band held in shared memory as a ring of Wc columns; NIO further warps write the
// columns the train has left behind back to global memory and fetch the ones the leading sweep needs next, concurrently
// with the arithmetic.  When the whole band fits the ring (small n) it is loaded once, never written back (only d, e
// are outputs), and the teams run one continuous pipeline over all sweeps instead of trains.
//
// Element (r, c), c <= r <= c + 2B - 1, lives at ring[(c mod Wc) * LD + (r - c)].  With LD = 2B the two access patterns
// used (fixed column, lanes over rows: stride 1; fixed row, lanes over columns: stride LD - 1, odd) are both free of
// shared-memory bank conflicts for 16-byte elements.
#include "bs_internal.cuh"

namespace bsk {

namespace {
constexpr int NIO = 4;  // I/O warps

__device__ __forceinline__ cplx shfl_c(cplx v, int src) {
  return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

// Sum over the B consecutive lanes that hold one vector (B = 8, 16 or 32); every lane of the group gets the same bits.
template <int B>
__device__ __forceinline__ double group_sum(double x) {
#pragma unroll
  for (int o = B / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

// LAPACK zlarfg on a vector spread over a group of B lanes (x valid for l < len; others must hold 0):
// H = I - tau v v^H, H^H x = beta e_1, beta real, v[0] = 1.  Returns v in x.
template <int B>
__device__ __forceinline__ void group_larfg(cplx &x, int len, int l, cplx &tau, double &beta) {
  const double mine = (l >= 1 && l < len) ? x.x * x.x + x.y * x.y : 0.0;
  const double ss = group_sum<B>(mine);
  const int base = (threadIdx.x & 31) & ~(B - 1);
  const cplx al = shfl_c(x, base);
  if (ss == 0.0 && al.y == 0.0) {
    tau = cmake(0.0, 0.0);
    beta = al.x;
    x = (l == 0) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
    return;
  }
  beta = -copysign(sqrt(al.x * al.x + al.y * al.y + ss), al.x);
  tau = cmake((beta - al.x) / beta, -al.y / beta);
  const double dr = al.x - beta, di = al.y, den = 1.0 / (dr * dr + di * di);
  const cplx scale = cmake(dr * den, -di * den);
  if (l == 0) x = cmake(1.0, 0.0);
  else if (l < len) x = cmul(x, scale);
  else x = cmake(0.0, 0.0);
}

// Team of 4B threads per sweep: thread (l, q), l = index inside the B x B block (row or column), q = quarter of the
// other dimension (QN = B/4 indices each).  Vectors (v, w, u, v2) are computed redundantly by the four q-replicas.
template <int B, int NQ>
__global__ void __launch_bounds__(NQ * B >= 128 ? 512 : 1024) bulge_kernel(int n, BatchRef AB, double *d, double *e, int G,
                                                                             int Wc, int inner) {
  constexpr int LD = 2 * B, TT = NQ * B, QN = B / NQ;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *ring = reinterpret_cast<cplx *>(smem_raw);
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *ab = batch_ptr(AB, cell, mi);
  double *dg = d + (size_t)z * n, *eg = e + (size_t)z * n;
  const int tid = threadIdx.x;
  const int ncomp = G * TT;
  const bool is_io = tid >= ncomp;
  const int io_tid = tid - ncomp, io_nt = blockDim.x - ncomp;
  const int team = tid / TT, tt = tid % TT, l = tt % B, q = tt / B;
  // team scratch behind the ring: vs, ws, tus, v2s (B each), red1, red2, red3 (NQ B each) complex per team
  cplx *ts = ring + (size_t)Wc * LD + (size_t)(is_io ? 0 : team) * (4 + 3 * NQ) * B;
  cplx *vs = ts, *ws = ts + B, *tus = ts + 2 * B, *v2s = ts + 3 * B;
  cplx *red1 = ts + 4 * B, *red2 = red1 + NQ * B, *red3 = red2 + NQ * B;
  auto qsum = [&](const cplx *red) {  // fixed order: identical bits in every replica
    cplx a = red[l];
#pragma unroll
    for (int qq = 1; qq < NQ; ++qq) a = cadd(a, red[qq * B + l]);
    return a;
  };
  auto team_bar = [&]() {
    if (TT == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;\n" ::"r"(team + 1), "r"(TT) : "memory");
  };
  const bool resident = n <= Wc;

  int wlo = 0, whi = 0;  // ring holds columns [wlo, whi)  (uniform over the CTA)
  auto slot_of = [&](int c) { return c % Wc; };
  // column ranges are copied as one flat index space so that every thread has several independent 16-byte
  // transfers in flight (cp.async: global -> shared without register staging)
  // Thread t of nt (nt a multiple of LD) moves element off = t % LD of the columns c0 + t / LD + j (nt / LD): the ring
  // slot is advanced incrementally and every thread keeps several independent 16-byte transfers in flight.
  auto io_load = [&](int c0, int c1, int t, int nt) {
    const int off = t % LD, cstep = nt / LD;
    int c = c0 + t / LD;
    if (c < c1) {
      int sl = slot_of(c);
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
      int sl = slot_of(c);
      const int sstep = cstep % Wc;
#pragma unroll 4
      for (; c < c1; c += cstep) {
        ab[(size_t)c * LD + off] = ring[(size_t)sl * LD + off];
        sl += sstep;
        if (sl >= Wc) sl -= Wc;
      }
    }
  };

  if (resident) {
    io_load(0, n, tid, blockDim.x);
    wlo = 0; whi = n;
    __syncthreads();
  }

  // per-team sweep state (identical in all threads of a team)
  int i = 0, k = 0, J = 0, L = 0;
  bool finished = true;
  cplx v = cmake(0.0, 0.0), tau = cmake(0.0, 0.0);
  // one step of sweep i (the whole team executes it)
  auto do_step = [&]() {
    // -------------------------------------------------------------------- one step of sweep i
    if (k == 0) {
      L = min(B, n - 1 - i);
      const cplx *ci = ring + (size_t)slot_of(i) * LD;
      cplx x = l < L ? ci[1 + l] : cmake(0.0, 0.0);
      double beta;
      group_larfg<B>(x, L, l, tau, beta);
      v = x;
      if (tt == 0) { eg[i] = beta; dg[i] = ci[0].x; }
      if (q == 0) vs[l] = v;
      team_bar();
    }
    const int sJ = slot_of(J);
    // element offsets of the ring columns this thread touches: its quarter (J + q QN + jj) and column J + l
    int cb[QN];
#pragma unroll
    for (int jj = 0; jj < QN; ++jj) {
      int sl = sJ + q * QN + jj;
      if (sl >= Wc) sl -= Wc;
      cb[jj] = sl * LD;
    }
    int mycb = sJ + l;
    if (mycb >= Wc) mycb -= Wc;
    mycb *= LD;
    const int cb0 = sJ * LD;
    const bool t_on = (tau.x != 0.0 || tau.y != 0.0);
    const int Jn = J + L, L2 = min(B, n - Jn);
    // P1: partial p = D v over this thread's quarter of the columns; P4: partial u = C v
    // (branch-free: every index is a valid ring address, invalid contributions are masked through v)
    cplx acc = cmake(0.0, 0.0), uacc = cmake(0.0, 0.0);
    if (t_on) {
#pragma unroll
      for (int jj = 0; jj < QN; ++jj) {
        const int c = q * QN + jj;
        cplx vc = vs[c];
        vc.x = c < L ? vc.x : 0.0;
        vc.y = c < L ? vc.y : 0.0;
        cplx a = ring[l >= c ? cb[jj] + l - c : mycb + c - l];  // lower part as stored, upper part mirrored
        a.y = l > c ? a.y : (l == c ? 0.0 : -a.y);
        cfma(acc, a, vc);
        cfma(uacc, ring[cb[jj] + max(L + l - c, 0)], vc);  // (negative only where vc is masked to zero)
      }
      acc.x = l < L ? acc.x : 0.0;
      acc.y = l < L ? acc.y : 0.0;
      uacc.x = l < L2 ? uacc.x : 0.0;
      uacc.y = l < L2 ? uacc.y : 0.0;
    }
    red1[q * B + l] = acc;
    red2[q * B + l] = uacc;
    team_bar();  // BAR1
    // P2 (w from p) and P5 (first column of C after the right-apply and the reflector that annihilates it) as one
    // straight-line block: the three lane reductions and the sqrt / divisions of the two chains overlap
    cplx p = cmul(tau, qsum(red1));
    const cplx u = qsum(red2);
    const cplx tu = cmul(tau, u);
    cplx x = csub(ring[cb0 + L + l], tu);  // conj(v[0]) = 1; always a valid ring address
    x.x = l < L2 ? x.x : 0.0;
    x.y = l < L2 ? x.y : 0.0;
    double sr = l < L ? p.x * v.x + p.y * v.y : 0.0;  // p^H v
    double si = l < L ? p.x * v.y - p.y * v.x : 0.0;
    double ss = l >= 1 ? x.x * x.x + x.y * x.y : 0.0;
#pragma unroll
    for (int o = B / 2; o > 0; o >>= 1) {
      sr += __shfl_xor_sync(0xffffffffu, sr, o);
      si += __shfl_xor_sync(0xffffffffu, si, o);
      ss += __shfl_xor_sync(0xffffffffu, ss, o);
    }
    const cplx alpha = cmul(cmake(-0.5 * tau.x, -0.5 * tau.y), cmake(sr, si));
    cplx w = p;
    cfma(w, alpha, v);
    // zlarfg, branch-free: no reflector when the block has a single row (L2 <= 1) or the column is already e_1-shaped
    const cplx al = shfl_c(x, (threadIdx.x & 31) & ~(B - 1));
    const bool norefl = L2 <= 1, trivial = norefl || (ss == 0.0 && al.y == 0.0);
    const double nrm = sqrt(al.x * al.x + al.y * al.y + ss);
    const double beta2 = trivial ? 1.0 : -copysign(nrm, al.x);
    const double ib = 1.0 / beta2;
    cplx tau2 = cmake((beta2 - al.x) * ib, -al.y * ib);
    tau2.x = trivial ? 0.0 : tau2.x;
    tau2.y = trivial ? 0.0 : tau2.y;
    const double dr = al.x - beta2, di = al.y;
    const double den = 1.0 / (dr * dr + di * di);
    cplx scale = cmake(dr * den, -di * den);
    scale.x = trivial ? 0.0 : scale.x;
    scale.y = trivial ? 0.0 : scale.y;
    cplx v2 = cmul(x, scale);
    v2.x = l == 0 ? 1.0 : v2.x;
    v2.y = l == 0 ? 0.0 : v2.y;
    if (q == 0 && l < L2) {
      cplx c00 = norefl ? x : cmake(trivial ? al.x : beta2, 0.0);
      ring[cb0 + L + l] = (l == 0) ? c00 : cmake(0.0, 0.0);
    }
    if (q == 0) { ws[l] = w; tus[l] = tu; v2s[l] = v2; }
    team_bar();  // BAR2
    // P3: D <- D - v w^H - w v^H on the lower triangle (all loads first, then all stores: no false dependences)
    if (t_on) {
      cplx av[QN];
#pragma unroll
      for (int jj = 0; jj < QN; ++jj) {
        const int c = q * QN + jj;
        av[jj] = ring[cb[jj] + max(l - c, 0)];
      }
#pragma unroll
      for (int jj = 0; jj < QN; ++jj) {
        const int c = q * QN + jj;
        cplx a = av[jj];
        cfms(a, v, cconj(ws[c]));
        cfms(a, w, cconj(vs[c]));
        a.y = l == c ? 0.0 : a.y;
        av[jj] = a;
      }
#pragma unroll
      for (int jj = 0; jj < QN; ++jj) {
        const int c = q * QN + jj;
        if (c <= l && l < L) ring[cb[jj] + (l - c)] = av[jj];
      }
    }
    if (L2 <= 0) {
      finished = true;
    } else {
      const bool t2_on = (tau2.x != 0.0 || tau2.y != 0.0);
      if (t_on || t2_on) {
        // P6/P7: thread = column c = l of C (1 <= c < L), rows of its quarter:
        //   t = C - (tau C v) v^H ; z = v2^H t ; C = t - v2 conj(tau2) z
        const bool mine = l >= 1 && l < L;
        const cplx vcj = cconj(v);
        cplx *pc = ring + (mine ? mycb + L - l : cb0 + L);
        cplx tv[QN];
        cplx zacc = cmake(0.0, 0.0);
#pragma unroll
        for (int jj = 0; jj < QN; ++jj) {
          const int r = q * QN + jj;
          cplx t = pc[r];
          cplx tur = tus[r], v2r = v2s[r];
          v2r.x = r < L2 ? v2r.x : 0.0;  // rows beyond the block do not contribute
          v2r.y = r < L2 ? v2r.y : 0.0;
          cfms(t, tur, vcj);
          cfmac(zacc, v2r, t);
          tv[jj] = t;
        }
        zacc.x = mine ? zacc.x : 0.0;
        zacc.y = mine ? zacc.y : 0.0;
        red3[q * B + l] = zacc;
        team_bar();  // BAR3
        const cplx zc = qsum(red3);
        const cplx f = cmul(cconj(tau2), zc);
#pragma unroll
        for (int jj = 0; jj < QN; ++jj) {
          const int r = q * QN + jj;
          cplx t = tv[jj];
          cfms(t, v2s[r], f);
          if (mine && r < L2) pc[r] = t;
        }
      }
      if (q == 0) vs[l] = v2;  // after BAR3 (or with P3 skipped): nobody still reads the old v
      v = v2; tau = tau2; J = Jn; L = L2; ++k;
    }
  };

  if (resident) {
    // The whole band is in shared memory: no trains, the teams run a continuous pipeline.  Sweep i starts at macro-step
    // start[i] = max(start[i-1] + 2, finish of sweep i-G) (two blocks behind its predecessor, and its team must be free).
    int *start = reinterpret_cast<int *>(ring + (size_t)Wc * LD + (size_t)G * (4 + 3 * NQ) * B);
    if (tid == 0) {
      for (int j = 0; j <= n - 2; ++j) {
        int st = j == 0 ? 0 : start[j - 1] + 2;
        if (j >= G) st = max(st, start[j - G] + (n - 1 - (j - G) + B - 1) / B);
        start[j] = st;
      }
    }
    __syncthreads();
    const int S = n >= 2 ? start[n - 2] + 1 : 0;  // the last sweep has a single step
    int next_i = team;
    for (int s = 0; s < S; ++s) {
      if (!is_io) {
        if (finished && next_i <= n - 2 && start[next_i] == s) {
          i = next_i; k = 0; J = i + 1; L = 0; finished = false;
          tau = cmake(0.0, 0.0);
        }
        if (!finished) {
          do_step();
          if (finished) next_i += G;
        }
      }
      __syncthreads();
    }
  } else {
    for (int t0 = 0; t0 < n - 1; t0 += G) {
      const int nvalid = min(G, n - 1 - t0);  // sweeps t0 .. t0+nvalid-1
      if (!resident) {
        // (re)position the window at the head of the band for this train
        const int need = min(n, t0 + 1 + B);
        if (t0 < wlo || t0 >= whi) {
          io_evict(max(wlo, t0), whi, tid, blockDim.x);  // columns < t0 are finished: never read again
          __syncthreads();
          io_load(t0, need, tid, blockDim.x);
          wlo = t0; whi = need;
        } else if (whi < need) {
          io_load(whi, need, tid, blockDim.x);
          whi = need;
        }
        __syncthreads();
      }
      i = t0 + team;
      const bool valid = !is_io && team < nvalid;
      k = 0; J = i + 1; L = 0;
      finished = !valid;
      v = cmake(0.0, 0.0); tau = cmake(0.0, 0.0);
      const int nsteps0 = (n - 1 - t0 + B - 1) / B;
      const int S = nsteps0 + 2 * (nvalid - 1);

      for (int s = 0; s < S; ++s) {
        if (!resident) {  // window bookkeeping (uniform): columns needed at macro-step s or later / at s+1
          int keep = n, hi = whi;
          for (int g = 0; g < nvalid; ++g) {
            const int ig = t0 + g, kg = s - 2 * g, ns = (n - 1 - ig + B - 1) / B;
            if (kg >= ns) continue;  // finished
            keep = min(keep, kg <= 0 ? ig : ig + 1 + kg * B);
            const int k1 = kg + 1;
            if (k1 >= 0 && k1 < ns) hi = max(hi, min(n, ig + 1 + (k1 + 1) * B));
          }
          keep = max(keep, wlo);
          if (is_io) {
            io_evict(max(wlo, t0 + nvalid), keep, io_tid, io_nt);  // columns < t0+nvalid are finished
            // the columns fetched now reuse ring slots of the columns written back just above (hi - wlo exceeds Wc by
            // up to B - G - 7), in general through another thread: all slot reads first
            asm volatile("bar.sync 15, %0;\n" ::"r"(NIO * 32) : "memory");
            io_load(whi, hi, io_tid, io_nt);
          }
          wlo = keep; whi = hi;
        }
        if (!finished && s >= 2 * team) do_step();
        __syncthreads();
      }
    }
  }
  // last diagonal entry
  if (tid == 0) {
    if (n >= 1) {
      const bool in_ring = (n - 1 >= wlo && n - 1 < whi);
      dg[n - 1] = in_ring ? ring[(size_t)slot_of(n - 1) * LD].x : ab[(size_t)(n - 1) * LD].x;
      eg[n - 1] = 0.0;
    }
  }
}

constexpr size_t BULGE_MAX_SMEM = 226 * 1024;
constexpr int bulge_gmax(int B, int NQ) {  // teams per CTA (G * TT + 128 I/O threads)
  return min(12, ((NQ * B >= 128 ? 512 : 1024) - NIO * 32) / (NQ * B));
}
constexpr bool bulge_fits(int n, int B, int NQ) {  // the whole band (n columns of 2B entries) beside the team scratch
  return (size_t)n * 2 * B * sizeof(cplx) + (size_t)bulge_gmax(B, NQ) * (4 + 3 * NQ) * B * sizeof(cplx) +
             (size_t)n * sizeof(int) <= BULGE_MAX_SMEM;
}

template <int B, int NQ>
void launch_bulge_t(int n, BatchRef AB, double *d, double *e, int nmat, int inner, bool streamed, cudaStream_t s) {
  constexpr int LD = 2 * B, TT = NQ * B;
  const size_t colbytes = (size_t)LD * sizeof(cplx);
  const int gmax = bulge_gmax(B, NQ);
  const size_t team_bytes = (size_t)(4 + 3 * NQ) * B * sizeof(cplx);
  const size_t max_smem = BULGE_MAX_SMEM;
  int G, Wc;
  if (streamed && n > 2 * 3 * B + 8) {  // BS_TRIDIAG_TWO_STAGE_STREAMED: the ring of three sweeps whatever n
    G = min(3, gmax);
    Wc = 2 * G * B + 8;
  } else if (bulge_fits(n, B, NQ)) {  // whole band resident
    Wc = max(n, 2 * B + 8);  // never fewer than a block pair of columns: the masked loads of a step stay inside the ring
    G = max(1, min(gmax, (n + 2 * B - 1) / (2 * B)));
  } else {
    G = (int)(((max_smem - gmax * team_bytes) / colbytes - 8) / (2 * B));
    G = max(1, min(G, gmax));
    Wc = 2 * G * B + 8;
  }
  const size_t smem = (size_t)Wc * colbytes + G * team_bytes + (Wc >= n ? (size_t)n * sizeof(int) : 0);
  static unsigned long long attr_mask = 0;
  ensure_dyn_smem(bulge_kernel<B, NQ>, 227 * 1024, attr_mask);
  // algorithmic work: ~n^2/(2B) steps of 48 B^2 real flops (hemv, rank-2, C v, right- and left-apply)
  KScope ks(KC_BULGE, 24.0 * n * (double)n * B * nmat, s);
  // the I/O warps only exist when the band is streamed through the ring
  bulge_kernel<B, NQ><<<nmat, G * TT + (Wc >= n ? 0 : NIO * 32), smem, s>>>(n, AB, d, e, G, Wc, inner);
}
}  // namespace

bool bulge_band_resident(int n, int b) { return bulge_fits(n, b >= 32 ? 32 : (b >= 16 ? 16 : 8), 4); }

// Band -> tridiagonal for every matrix of the batch.  b must be 8, 16 or 32.
void launch_sb2st(int n, int b, BatchRef AB, double *d, double *e, int ncells, int inner, cudaStream_t s, bool streamed) {
  const int nmat = ncells * inner;
  if (b == 8) launch_bulge_t<8, 4>(n, AB, d, e, nmat, inner, streamed, s);
  else if (b == 16) launch_bulge_t<16, 4>(n, AB, d, e, nmat, inner, streamed, s);
  else launch_bulge_t<32, 4>(n, AB, d, e, nmat, inner, streamed, s);
}

}  // namespace bsk
