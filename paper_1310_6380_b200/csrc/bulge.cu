// S6, stage 2: Hermitian band (width B, lower storage with bulge space, ldab = 2B) -> real symmetric tridiagonal by
// Householder bulge chasing (column-wise elimination, Schwarz / Lang).  DESIGN.md section 5 (S6, stage 2).
//
// One CTA per matrix.  Sweep i annihilates column i below the sub-diagonal and chases the bulge down the band in steps
// of B columns; step k of sweep i touches columns [i+1+kB, i+1+(k+1)B) only, so sweep i+1 can run two steps behind sweep i.
// A "train" of G consecutive sweeps is executed by G warps in lock step (warp g does step s-2g at macro-step s) on a
// window of the band held in shared memory as a ring of Wc columns; NIO further warps write the columns the train has
// left behind back to global memory and fetch the ones the leading sweep needs next, concurrently with the arithmetic.
// When the whole band fits the ring (small n) it is loaded once and never written back (only d, e are outputs).
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

// LAPACK zlarfg on a vector spread over the lanes (x valid for lane < len; others must hold 0):
// H = I - tau v v^H, H^H x = beta e_1, beta real, v[0] = 1.  Returns v in x.
__device__ __forceinline__ void warp_larfg(cplx &x, int len, int lane, cplx &tau, double &beta) {
  const double mine = (lane >= 1 && lane < len) ? x.x * x.x + x.y * x.y : 0.0;
  const double ss = warp_sum(mine);
  const cplx al = shfl_c(x, 0);
  if (ss == 0.0 && al.y == 0.0) {
    tau = cmake(0.0, 0.0);
    beta = al.x;
    x = (lane == 0) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
    return;
  }
  beta = -copysign(sqrt(al.x * al.x + al.y * al.y + ss), al.x);
  tau = cmake((beta - al.x) / beta, -al.y / beta);
  const double dr = al.x - beta, di = al.y, den = 1.0 / (dr * dr + di * di);
  const cplx scale = cmake(dr * den, -di * den);
  if (lane == 0) x = cmake(1.0, 0.0);
  else if (lane < len) x = cmul(x, scale);
  else x = cmake(0.0, 0.0);
}

template <int B>
__global__ void __launch_bounds__(512) bulge_kernel(int n, BatchRef AB, double *d, double *e, int G, int Wc, int inner) {
  constexpr int LD = 2 * B;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *ring = reinterpret_cast<cplx *>(smem_raw);
  const int z = blockIdx.x, cell = z / inner, mi = z % inner;
  cplx *ab = batch_ptr(AB, cell, mi);
  double *dg = d + (size_t)z * n, *eg = e + (size_t)z * n;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool is_io = warp >= G;
  const int io_tid = tid - G * 32, io_nt = NIO * 32;
  const bool resident = n <= Wc;

  int wlo = 0, whi = 0;  // ring holds columns [wlo, whi)  (uniform over the CTA)
  auto slot_of = [&](int c) { return c % Wc; };
  auto io_load = [&](int c0, int c1, int t, int nt) {
    for (int c = c0; c < c1; ++c) {
      const cplx *src = ab + (size_t)c * LD;
      cplx *dst = ring + (size_t)slot_of(c) * LD;
      for (int q = t; q < LD; q += nt) dst[q] = src[q];
    }
  };
  auto io_evict = [&](int c0, int c1, int t, int nt) {
    for (int c = c0; c < c1; ++c) {
      cplx *dst = ab + (size_t)c * LD;
      const cplx *src = ring + (size_t)slot_of(c) * LD;
      for (int q = t; q < LD; q += nt) dst[q] = src[q];
    }
  };

  if (resident) {
    io_load(0, n, tid, blockDim.x);
    wlo = 0; whi = n;
    __syncthreads();
  }

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
    // per-warp sweep state
    const int i = t0 + warp;
    const bool valid = !is_io && warp < nvalid;
    int k = 0, J = i + 1, L = 0;
    bool finished = !valid;
    cplx v = cmake(0.0, 0.0), tau = cmake(0.0, 0.0);
    const int nsteps0 = (n - 1 - t0 + B - 1) / B;
    const int S = nsteps0 + 2 * (nvalid - 1);

    for (int s = 0; s < S; ++s) {
      if (is_io) {
        if (!resident) {
          // columns still needed at macro-step s or later / needed at macro-step s+1
          int keep = n, hi = whi;
          for (int g = 0; g < nvalid; ++g) {
            const int ig = t0 + g, kg = s - 2 * g, ns = (n - 1 - ig + B - 1) / B;
            if (kg >= ns) continue;  // finished
            keep = min(keep, kg <= 0 ? ig : ig + 1 + kg * B);
            const int k1 = kg + 1;
            if (k1 >= 0 && k1 < ns) hi = max(hi, min(n, ig + 1 + (k1 + 1) * B));
          }
          keep = max(keep, wlo);
          io_evict(max(wlo, t0 + nvalid), keep, io_tid, io_nt);  // columns < t0+nvalid are finished
          io_load(whi, hi, io_tid, io_nt);
          wlo = keep; whi = hi;
        }
      } else {
        if (!resident) {  // mirror the window bookkeeping (uniform values; compute warps only need them at train change)
          int keep = n, hi = whi;
          for (int g = 0; g < nvalid; ++g) {
            const int ig = t0 + g, kg = s - 2 * g, ns = (n - 1 - ig + B - 1) / B;
            if (kg >= ns) continue;
            keep = min(keep, kg <= 0 ? ig : ig + 1 + kg * B);
            const int k1 = kg + 1;
            if (k1 >= 0 && k1 < ns) hi = max(hi, min(n, ig + 1 + (k1 + 1) * B));
          }
          wlo = max(keep, wlo); whi = hi;
        }
        if (!finished && s >= 2 * warp) {
          // ------------------------------------------------------------------ one step of sweep i
          if (k == 0) {
            L = min(B, n - 1 - i);
            const cplx *ci = ring + (size_t)slot_of(i) * LD;
            cplx x = lane < L ? ci[1 + lane] : cmake(0.0, 0.0);
            double beta;
            warp_larfg(x, L, lane, tau, beta);
            v = x;
            if (lane == 0) { eg[i] = beta; dg[i] = ci[0].x; }
          }
          const int sJ = slot_of(J);
          auto col = [&](int cc) {  // ring column J + cc
            int sl = sJ + cc;
            if (sl >= Wc) sl -= Wc;
            return ring + (size_t)sl * LD;
          };
          if (tau.x != 0.0 || tau.y != 0.0) {
            // two-sided update of the diagonal block D = A[J:J+L, J:J+L]:  D <- H^H D H  (zhetd2 form)
            cplx p = cmake(0.0, 0.0);
            for (int c = 0; c < L; ++c) {
              const cplx vc = shfl_c(v, c);
              if (lane < L) {
                cplx a;
                if (lane >= c) { a = col(c)[lane - c]; if (lane == c) a.y = 0.0; }
                else a = cconj(col(lane)[c - lane]);
                cfma(p, a, vc);
              }
            }
            p = cmul(tau, p);
            const double sr = warp_sum(lane < L ? p.x * v.x + p.y * v.y : 0.0);  // p^H v
            const double si = warp_sum(lane < L ? p.x * v.y - p.y * v.x : 0.0);
            const cplx alpha = cmul(cmake(-0.5 * tau.x, -0.5 * tau.y), cmake(sr, si));
            cplx w = p;
            cfma(w, alpha, v);
            for (int c = 0; c < L; ++c) {
              const cplx vc = shfl_c(v, c), wc = shfl_c(w, c);
              if (lane >= c && lane < L) {
                cplx *pa = col(c) + (lane - c);
                cplx a = *pa;
                cfms(a, v, cconj(wc));
                cfms(a, w, cconj(vc));
                if (lane == c) a.y = 0.0;
                *pa = a;
              }
            }
          }
          const int Jn = J + L, L2 = min(B, n - Jn);
          if (L2 <= 0) {
            finished = true;
          } else {
            // C = A[Jn:Jn+L2, J:J+L]:  C <- C H, new reflector from C[:,0], C[:,1:] <- H'^H C[:,1:]
            cplx u = cmake(0.0, 0.0);
            const bool t_on = (tau.x != 0.0 || tau.y != 0.0);
            if (t_on) {
              for (int c = 0; c < L; ++c) {
                const cplx vc = shfl_c(v, c);
                if (lane < L2) cfma(u, col(c)[L + lane - c], vc);
              }
            }
            const cplx tu = cmul(tau, u);  // row-wise tau (C v)
            cplx x = cmake(0.0, 0.0);
            if (lane < L2) { x = col(0)[L + lane]; x = csub(x, tu); }  // conj(v[0]) = 1
            cplx tau2 = cmake(0.0, 0.0), v2;
            if (L2 > 1) {
              double beta2;
              warp_larfg(x, L2, lane, tau2, beta2);
              v2 = x;
              if (lane < L2) col(0)[L + lane] = (lane == 0) ? cmake(beta2, 0.0) : cmake(0.0, 0.0);
            } else {
              if (lane == 0) col(0)[L] = x;
              v2 = (lane == 0) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
            }
            const bool t2_on = (tau2.x != 0.0 || tau2.y != 0.0);
            if (t_on || t2_on) {
              // lane = column c of C (1 <= c < L)
              const bool mine = lane >= 1 && lane < L;
              const cplx vcj = cconj(v);
              cplx *pc = col(mine ? lane : 0) + (L - (mine ? lane : 0));  // &C(0, c)
              cplx zacc = cmake(0.0, 0.0);
              for (int r = 0; r < L2; ++r) {
                const cplx tur = shfl_c(tu, r), v2r = shfl_c(v2, r);
                if (mine) {
                  cplx t = pc[r];
                  cfms(t, tur, vcj);
                  cfmac(zacc, v2r, t);
                  pc[r] = t;
                }
              }
              if (t2_on) {
                const cplx f = cmul(cconj(tau2), zacc);
                for (int r = 0; r < L2; ++r) {
                  const cplx v2r = shfl_c(v2, r);
                  if (mine) {
                    cplx t = pc[r];
                    cfms(t, v2r, f);
                    pc[r] = t;
                  }
                }
              }
            }
            v = v2; tau = tau2; J = Jn; L = L2; ++k;
          }
        }
      }
      __syncthreads();
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

template <int B>
void launch_bulge_t(int n, BatchRef AB, double *d, double *e, int nmat, int inner, cudaStream_t s) {
  constexpr int LD = 2 * B;
  const size_t colbytes = (size_t)LD * sizeof(cplx);
  const size_t max_smem = 220 * 1024;
  int G, Wc;
  if ((size_t)n * colbytes <= max_smem) {  // whole band resident
    Wc = n;
    G = max(1, min(12, (n + 2 * B - 1) / (2 * B)));
  } else {
    G = (int)((max_smem / colbytes - 8) / (2 * B));
    G = max(1, min(G, 12));
    Wc = 2 * G * B + 8;
  }
  const size_t smem = (size_t)Wc * colbytes;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(bulge_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    attr_done = true;
  }
  KScope ks(KC_BULGE, 0.0, s);
  bulge_kernel<B><<<nmat, (G + NIO) * 32, smem, s>>>(n, AB, d, e, G, Wc, inner);
}
}  // namespace

// Band -> tridiagonal for every matrix of the batch.  b must be 8, 16 or 32.
void launch_sb2st(int n, int b, BatchRef AB, double *d, double *e, int ncells, int inner, cudaStream_t s) {
  const int nmat = ncells * inner;
  if (b == 8) launch_bulge_t<8>(n, AB, d, e, nmat, inner, s);
  else if (b == 16) launch_bulge_t<16>(n, AB, d, e, nmat, inner, s);
  else launch_bulge_t<32>(n, AB, d, e, nmat, inner, s);
}

}  // namespace bsk
