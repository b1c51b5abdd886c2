// S1 (shape-integral table) and S2 (expansion to Phi, R).  PAPER.md:140-173 (eq. 17-20) with the exact polygon
// integral in place of the centroid rule (eq. 12/22); DESIGN.md sections 3 (R1: entries depend only on the index
// difference) and 5.
#include "bs_internal.cuh"

namespace bsk {

static constexpr double kPi = 3.14159265358979323846264338327950288;

// One CTA (8 warps) per index difference D in the half plane {D1>0} u {D1==0, D2>=0}; the warps split the edges, lanes
// stride over a warp's slice, and the 8 x 32 partial sums are reduced in a fixed order (deterministic).
//   T_c(D) = (-i/|q|^2) sum_edges w_c[phase(e)] (q x e) exp(i q.m_e) j0(q.e/2),   q = D1 q^1 + D2 q^2,
// and T_c(0) = sum_p w_c[p] area_p.  The phase q.m and the argument of j0 are evaluated in FRACTIONAL coordinates
// (q.x = 2 pi (D1 H1 + D2 H2) with integer D), so sincospi/sinpi reduce the argument exactly.
__global__ void __launch_bounds__(256) table_kernel(const Geometry *__restrict__ geos, int Mt, BatchRef table, int centroid_rule) {
  __shared__ double part[8][14];
  const int cell = blockIdx.y;
  const Geometry g = geos[cell];
  const int L = 4 * Mt + 1;
  const int L2 = L * L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int flat = blockIdx.x + (L2 - 1) / 2;
  const int D1 = flat / L - 2 * Mt;
  const int D2 = flat % L - 2 * Mt;
  cplx *T = batch_ptr(table, cell, 0);

  double accr[7], acci[7];
#pragma unroll
  for (int c = 0; c < 7; ++c) accr[c] = acci[c] = 0.0;

  if (D1 == 0 && D2 == 0) {
    for (int p = threadIdx.x; p < g.P; p += 256) {
      const double a = g.area[p];
#pragma unroll
      for (int c = 0; c < 7; ++c) accr[c] = fma(g.w[c * g.P + p], a, accr[c]);
    }
  } else if (centroid_rule) {
    // PAPER.md:106 (eq. 12) / :213 (eq. 22): I_p(q) ~ A_p exp(i q.c_p), the paper's one-point rule per mesh element
    for (int p = threadIdx.x; p < g.P; p += 256) {
      const double phi = fma((double)D1, g.area[g.P + p], (double)D2 * g.area[2 * g.P + p]);  // q.c / (2 pi)
      double sn, cs;
      sincospi(2.0 * phi, &sn, &cs);
      const double a = g.area[p];
      const double tr = a * cs, ti = a * sn;
#pragma unroll
      for (int c = 0; c < 7; ++c) {
        const double w = g.w[c * g.P + p];
        accr[c] = fma(w, tr, accr[c]);
        acci[c] = fma(w, ti, acci[c]);
      }
    }
  } else {
    const double qx = D1 * g.Q[0] + D2 * g.Q[2];
    const double qy = D1 * g.Q[1] + D2 * g.Q[3];
    const int ne = g.nedge, nes = g.nes;
    const double *mh1 = g.edge, *mh2 = g.edge + nes, *eh1 = g.edge + 2 * nes, *eh2 = g.edge + 3 * nes;
    const double *ex = g.edge + 4 * nes, *ey = g.edge + 5 * nes;
    for (int e = threadIdx.x; e < ne; e += 256) {
      const double phi = fma((double)D1, mh1[e], (double)D2 * mh2[e]);  // q.m / (2 pi)
      const double u = fma((double)D1, eh1[e], (double)D2 * eh2[e]);    // q.e / (2 pi)  ->  q.e/2 = pi u
      double sn, cs;
      sincospi(2.0 * phi, &sn, &cs);
      const double j0 = (u == 0.0) ? 1.0 : sinpi(u) / (kPi * u);
      const double f = (qx * ey[e] - qy * ex[e]) * j0;
      const double tr = f * cs, ti = f * sn;
      const int p = g.ephase[e];
#pragma unroll
      for (int c = 0; c < 7; ++c) {
        const double w = g.w[c * g.P + p];
        accr[c] = fma(w, tr, accr[c]);
        acci[c] = fma(w, ti, acci[c]);
      }
    }
  }
#pragma unroll
  for (int c = 0; c < 7; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      accr[c] += __shfl_xor_sync(0xffffffffu, accr[c], o);
      acci[c] += __shfl_xor_sync(0xffffffffu, acci[c], o);
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int c = 0; c < 7; ++c) { part[warp][2 * c] = accr[c]; part[warp][2 * c + 1] = acci[c]; }
  }
  __syncthreads();
  if (threadIdx.x < 7) {
    const int c = threadIdx.x;
    double sr = 0.0, si = 0.0;
    for (int w = 0; w < 8; ++w) { sr += part[w][2 * c]; si += part[w][2 * c + 1]; }
    if (D1 == 0 && D2 == 0) {
      T[(size_t)c * L2 + flat] = cmake(sr, 0.0);
    } else if (centroid_rule) {
      T[(size_t)c * L2 + flat] = cmake(sr, si);
      T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(sr, -si);
    } else {
      const double qx = D1 * g.Q[0] + D2 * g.Q[2];
      const double qy = D1 * g.Q[1] + D2 * g.Q[3];
      const double inv = 1.0 / (qx * qx + qy * qy);
      // (-i) * (ar + i ai) = ai - i ar
      const double re = si * inv, im = -sr * inv;
      T[(size_t)c * L2 + flat] = cmake(re, im);
      T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(re, -im);  // T(-D) = conj T(D): Phi, R exactly Hermitian
    }
  }
}

// ---------------------------------------------------------------------------------------------- S1 with TMA staging
// The same table, DPB index differences per CTA (one warp each), with the phase geometry and properties staged in shared
// memory by 1-D bulk TMA copies (cp.async.bulk, completion on an mbarrier): the weights w[7][P] and the areas once, the
// edge arrays in chunks of EC edges, double-buffered so that the copy of chunk i+1 runs under the arithmetic of chunk i.
// (north_star: "phase geometry and properties staged in shared memory via TMA".)
namespace {
constexpr int DPB = 16, EC = 1024;  // at most DPB index differences (warps) per CTA; edges per staged chunk
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__host__ __device__ __forceinline__ unsigned up16(unsigned b) { return (b + 15u) & ~15u; }
}  // namespace

size_t table_tma_smem(int P) {  // w, area, two edge chunks (6 arrays + phase indices), barriers, partial sums of Delta = 0
  return up16(7u * P * 8u) + up16(P * 8u) + 2 * (6 * EC * 8 + EC * 4) + 64;
}

__global__ void __launch_bounds__(DPB * 32) table_tma_kernel(const Geometry *__restrict__ geos, int Mt, BatchRef table) {
  extern __shared__ __align__(128) unsigned char tsm[];
  const int cell = blockIdx.y;
  const Geometry g = geos[cell];
  const int L = 4 * Mt + 1, L2 = L * L, nhalf = (L2 + 1) / 2;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int P = g.P, ne = g.nedge, nes = g.nes;
  double *ws = reinterpret_cast<double *>(tsm);                                   // [7][P]
  double *as = reinterpret_cast<double *>(tsm + up16(7u * P * 8u));               // [P]
  unsigned char *ebase = tsm + up16(7u * P * 8u) + up16(P * 8u);
  const size_t cbytes = 6 * EC * 8 + EC * 4;
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(ebase + 2 * cbytes);  // [0]: w + area, [1], [2]: chunks
  const int nchunk = (ne + EC - 1) / EC;
  auto issue_chunk = [&](int ch) {  // thread 0
    const int e0 = ch * EC, cnt = min(EC, ne - e0), buf = ch & 1;
    unsigned char *dst = ebase + buf * cbytes;
    const unsigned bd = up16(cnt * 8u), bi = up16(cnt * 4u);
    mbar_expect_tx(&bars[1 + buf], 6 * bd + bi);
    for (int k = 0; k < 6; ++k) bulk_g2s(dst + k * EC * 8, g.edge + (size_t)k * nes + e0, bd, &bars[1 + buf]);
    bulk_g2s(dst + 6 * EC * 8, g.ephase + e0, bi, &bars[1 + buf]);
  };
  if (threadIdx.x == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_init(&bars[2], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    mbar_expect_tx(&bars[0], up16(7u * P * 8u) + up16(P * 8u));
    bulk_g2s(ws, g.w, up16(7u * P * 8u), &bars[0]);
    bulk_g2s(as, g.area, up16(P * 8u), &bars[0]);
    issue_chunk(0);
  }
  __syncthreads();
  const int dh = blockIdx.x * (blockDim.x >> 5) + warp;  // this warp's index difference (half plane)
  const bool active = dh < nhalf;
  const int flat = dh + (L2 - 1) / 2;
  const int D1 = flat / L - 2 * Mt, D2 = flat % L - 2 * Mt;
  const double qx = D1 * g.Q[0] + D2 * g.Q[2], qy = D1 * g.Q[1] + D2 * g.Q[3];
  double accr[7], acci[7];
#pragma unroll
  for (int c = 0; c < 7; ++c) accr[c] = acci[c] = 0.0;
  mbar_wait(&bars[0], 0);
  if (active && D1 == 0 && D2 == 0) {
    for (int p = lane; p < P; p += 32) {
      const double a = as[p];
#pragma unroll
      for (int c = 0; c < 7; ++c) accr[c] = fma(ws[c * P + p], a, accr[c]);
    }
  }
  for (int ch = 0; ch < nchunk; ++ch) {
    const int buf = ch & 1, e0 = ch * EC, cnt = min(EC, ne - e0);
    if (threadIdx.x == 0 && ch + 1 < nchunk) issue_chunk(ch + 1);  // (its buffer was released by the barrier that ended chunk ch - 1)
    mbar_wait(&bars[1 + buf], (ch >> 1) & 1);
    if (active && !(D1 == 0 && D2 == 0)) {
      const double *eb = reinterpret_cast<const double *>(ebase + buf * cbytes);
      const int *ep = reinterpret_cast<const int *>(ebase + buf * cbytes + 6 * EC * 8);
      for (int e = lane; e < cnt; e += 32) {
        const double phi = fma((double)D1, eb[e], (double)D2 * eb[EC + e]);              // q.m / (2 pi)
        const double u = fma((double)D1, eb[2 * EC + e], (double)D2 * eb[3 * EC + e]);  // q.e / (2 pi)
        double sn, cs;
        sincospi(2.0 * phi, &sn, &cs);
        const double j0 = (u == 0.0) ? 1.0 : sinpi(u) / (kPi * u);
        const double f = (qx * eb[5 * EC + e] - qy * eb[4 * EC + e]) * j0;
        const double tr = f * cs, ti = f * sn;
        const int p = ep[e];
#pragma unroll
        for (int c = 0; c < 7; ++c) {
          const double w = ws[c * P + p];
          accr[c] = fma(w, tr, accr[c]);
          acci[c] = fma(w, ti, acci[c]);
        }
      }
    }
    __syncthreads();  // every warp is done with this buffer: it may be refilled (chunk ch + 2)
  }
  if (!active) return;
#pragma unroll
  for (int c = 0; c < 7; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      accr[c] += __shfl_xor_sync(0xffffffffu, accr[c], o);
      acci[c] += __shfl_xor_sync(0xffffffffu, acci[c], o);
    }
  }
  cplx *T = batch_ptr(table, cell, 0);
  if (lane < 7) {
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int c = 0; c < 7; ++c) {
      sr = lane == c ? accr[c] : sr;
      si = lane == c ? acci[c] : si;
    }
    const int c = lane;
    if (D1 == 0 && D2 == 0) {
      T[(size_t)c * L2 + flat] = cmake(sr, 0.0);
    } else {
      const double inv = 1.0 / (qx * qx + qy * qy);
      const double re = si * inv, im = -sr * inv;  // (-i) (sr + i si) / |q|^2
      T[(size_t)c * L2 + flat] = cmake(re, im);
      T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(re, -im);  // T(-D) = conj T(D): Phi, R exactly Hermitian
    }
  }
}


// ---------------------------------------------------------------------------------------------- S1 with separable phases
// The index differences form a lattice, q_D = D1 q^1 + D2 q^2, so the two transcendental factors of an edge term split
// into factors that depend on (edge, D1) and (edge, D2) only:
//   exp(i q.m)  = exp(2 pi i D1 mh1) exp(2 pi i D2 mh2),      sin(q.e / 2) = Im[ exp(pi i D1 eh1) exp(pi i D2 eh2) ].
// edge_phasor_kernel evaluates the four families once per (edge, d), d = -2Mt .. 2Mt (4 L nedge sincospi instead of
// L^2 nedge sincospi + sinpi), into a table that stays in L2; table_sep_kernel forms every term with two complex
// products.  Accuracy: a product of two correctly rounded unit phasors has an ABSOLUTE error of ~2e-16, which is what the
// phase factor needs; sin(q.e/2) is divided by q.e/2, so for |q.e / 2 pi| < 2^-10 (q almost perpendicular to the edge,
// including the cases where rounding leaves 1e-17 in place of an exact zero) the kernel calls sinpi directly: the
// relative error of j0 stays below 1e-13 everywhere.  A CTA takes a TA x TB tile of (D1, D2), one warp per index
// difference: its (TA + TB) rows of each family are shared by the warps through L1.  Weights, areas and the edge
// arrays are staged in shared memory by bulk TMA copies as in table_tma_kernel.
__global__ void __launch_bounds__(128) edge_phasor_kernel(const Geometry *__restrict__ geos, int Mt, BatchRef scratch) {
  const int cell = blockIdx.z;
  const Geometry g = geos[cell];
  const int L = 4 * Mt + 1, nes = g.nes;
  const int e = blockIdx.x * blockDim.x + threadIdx.x, di = blockIdx.y;
  if (e >= g.nedge) return;
  const double d = (double)(di - 2 * Mt);
  cplx *tab = batch_ptr(scratch, cell, 0);
  const size_t fam = (size_t)L * nes, at = (size_t)di * nes + e;
  double sn, cs;
  sincospi(2.0 * (d * g.edge[e]), &sn, &cs);
  tab[at] = cmake(cs, sn);
  sincospi(2.0 * (d * g.edge[nes + e]), &sn, &cs);
  tab[fam + at] = cmake(cs, sn);
  sincospi(d * g.edge[2 * (size_t)nes + e], &sn, &cs);
  tab[2 * fam + at] = cmake(cs, sn);
  sincospi(d * g.edge[3 * (size_t)nes + e], &sn, &cs);
  tab[3 * fam + at] = cmake(cs, sn);
}

size_t table_sep_smem(int P) {  // w, area, two edge chunks (eh1, eh2, ex, ey + phase indices), barriers, partial sums
  return up16(7u * P * 8u) + up16(P * 8u) + 2 * (4 * EC * 8 + EC * 4) + 64 + DPB * 28 * 8;
}

// One PAIR of index differences (D1, +D2), (D1, -D2), D1, D2 >= 0, per two warps (each takes every other group of 32
// edges): the members share the four table loads, the edge data, the seven weights and the four real products of
// each phasor pair (cos/sin of a sum and of a difference), which halves the memory instructions per term.
__global__ void __launch_bounds__(DPB * 32) table_sep_kernel(const Geometry *__restrict__ geos, int Mt, BatchRef table,
                                                             BatchRef scratch, int TA, int TB) {
  extern __shared__ __align__(128) unsigned char tsm[];
  const int cell = blockIdx.y;
  const Geometry g = geos[cell];
  const int L = 4 * Mt + 1, L2 = L * L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int P = g.P, ne = g.nedge, nes = g.nes;
  double *ws = reinterpret_cast<double *>(tsm);                                   // [7][P]
  double *as = reinterpret_cast<double *>(tsm + up16(7u * P * 8u));               // [P]
  unsigned char *ebase = tsm + up16(7u * P * 8u) + up16(P * 8u);
  const size_t cbytes = 4 * EC * 8 + EC * 4;
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(ebase + 2 * cbytes);  // [0]: w + area, [1], [2]: chunks
  double *part = reinterpret_cast<double *>(ebase + 2 * cbytes + 64);                      // [warps][28]
  const int nchunk = (ne + EC - 1) / EC;
  auto issue_chunk = [&](int ch) {  // thread 0
    const int e0 = ch * EC, cnt = min(EC, ne - e0), buf = ch & 1;
    unsigned char *dst = ebase + buf * cbytes;
    const unsigned bd = up16(cnt * 8u), bi = up16(cnt * 4u);
    mbar_expect_tx(&bars[1 + buf], 4 * bd + bi);
    for (int k = 0; k < 4; ++k) bulk_g2s(dst + k * EC * 8, g.edge + (size_t)(k + 2) * nes + e0, bd, &bars[1 + buf]);
    bulk_g2s(dst + 4 * EC * 8, g.ephase + e0, bi, &bars[1 + buf]);
  };
  if (threadIdx.x == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_init(&bars[2], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    mbar_expect_tx(&bars[0], up16(7u * P * 8u) + up16(P * 8u));
    bulk_g2s(ws, g.w, up16(7u * P * 8u), &bars[0]);
    bulk_g2s(as, g.area, up16(P * 8u), &bars[0]);
    issue_chunk(0);
  }
  __syncthreads();
  // tile of pairs: D1 in [0, 2Mt], D2 in [0, 2Mt]
  const int n1 = 2 * Mt + 1, tb_count = (n1 + TB - 1) / TB;
  const int pw = warp >> 1, half = warp & 1;
  const int D1 = (blockIdx.x / tb_count) * TA + pw / TB, D2 = (blockIdx.x % tb_count) * TB + pw % TB;
  const bool active = D1 <= 2 * Mt && D2 <= 2 * Mt;
  const bool origin = D1 == 0 && D2 == 0;
  const bool minus = D1 > 0 && D2 > 0;  // (D1, -D2) is a member of the half plane of its own (else: the conjugate / the same)
  const double qxp = D1 * g.Q[0] + D2 * g.Q[2], qyp = D1 * g.Q[1] + D2 * g.Q[3];
  const double qxm = D1 * g.Q[0] - D2 * g.Q[2], qym = D1 * g.Q[1] - D2 * g.Q[3];
  const cplx *tab = batch_ptr(scratch, cell, 0);
  const size_t fam = (size_t)L * nes;
  const double2 *r1 = reinterpret_cast<const double2 *>(tab) + (size_t)(active ? D1 + 2 * Mt : 0) * nes;
  const double2 *r2 = reinterpret_cast<const double2 *>(tab) + fam + (size_t)(active ? D2 + 2 * Mt : 0) * nes;
  const double2 *r3 = r1 + 2 * fam, *r4 = r2 + 2 * fam;
  double apr[7], api[7], amr[7], ami[7];
#pragma unroll
  for (int c = 0; c < 7; ++c) apr[c] = api[c] = amr[c] = ami[c] = 0.0;
  mbar_wait(&bars[0], 0);
  if (active && origin) {
    for (int p = half * 32 + lane; p < P; p += 64) {
      const double a = as[p];
#pragma unroll
      for (int c = 0; c < 7; ++c) apr[c] = fma(ws[c * P + p], a, apr[c]);
    }
  }
  // sinc(pi u) = sin(pi u) / (pi u) from the product form sp of sin(pi u); see the header comment for the two guards
  auto sinc_of = [&](double u, double sp) {
    if (fabs(u) < 0x1p-10) sp = sinpi(u);
    const double y = kPi * u;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
    r = fma(r, fma(-y, r, 1.0), r);
    r = fma(r, fma(-y, r, 1.0), r);
    return (u == 0.0) ? 1.0 : sp * r;
  };
  for (int ch = 0; ch < nchunk; ++ch) {
    const int buf = ch & 1, e0 = ch * EC, cnt = min(EC, ne - e0);
    if (threadIdx.x == 0 && ch + 1 < nchunk) issue_chunk(ch + 1);  // (its buffer was released by the barrier that ended chunk ch - 1)
    mbar_wait(&bars[1 + buf], (ch >> 1) & 1);
    if (active && !origin) {
      const double *eb = reinterpret_cast<const double *>(ebase + buf * cbytes);
      const int *ep = reinterpret_cast<const int *>(ebase + buf * cbytes + 4 * EC * 8);
      // two edges per lane and pass: their eight table loads are issued before the first is used
      for (int eb0 = half * 32 + lane; eb0 < cnt; eb0 += 128) {
        double2 p1[2], p2[2], h1[2], h2[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int e = min(eb0 + 64 * k, cnt - 1);
          p1[k] = __ldg(r1 + e0 + e);  // (cos, sin)(2 pi D1 mh1)
          p2[k] = __ldg(r2 + e0 + e);  // (cos, sin)(2 pi D2 mh2)
          h1[k] = __ldg(r3 + e0 + e);  // (cos, sin)(pi D1 eh1)
          h2[k] = __ldg(r4 + e0 + e);  // (cos, sin)(pi D2 eh2)
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int e = eb0 + 64 * k;
          if (e >= cnt) break;
          const double t1 = (double)D1 * eb[e], t2 = (double)D2 * eb[EC + e];  // q.e / (2 pi) = t1 +- t2
          const double cc = p1[k].x * p2[k].x, ss = p1[k].y * p2[k].y, sc = p1[k].y * p2[k].x, cs = p1[k].x * p2[k].y;
          const double ba = h1[k].y * h2[k].x, ab = h1[k].x * h2[k].y;
          const double exv = eb[2 * EC + e], eyv = eb[3 * EC + e];
          const int p = ep[e];
          const double fp = (qxp * eyv - qyp * exv) * sinc_of(t1 + t2, ba + ab);
          const double trp = fp * (cc - ss), tip = fp * (sc + cs);
          double trm = 0.0, tim = 0.0;
          if (minus) {
            const double fm = (qxm * eyv - qym * exv) * sinc_of(t1 - t2, ba - ab);
            trm = fm * (cc + ss);
            tim = fm * (sc - cs);
          }
#pragma unroll
          for (int c = 0; c < 7; ++c) {
            const double w = ws[c * P + p];
            apr[c] = fma(w, trp, apr[c]);
            api[c] = fma(w, tip, api[c]);
            amr[c] = fma(w, trm, amr[c]);
            ami[c] = fma(w, tim, ami[c]);
          }
        }
      }
    }
    __syncthreads();  // every warp is done with this buffer: it may be refilled (chunk ch + 2)
  }
#pragma unroll
  for (int c = 0; c < 7; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      apr[c] += __shfl_xor_sync(0xffffffffu, apr[c], o);
      api[c] += __shfl_xor_sync(0xffffffffu, api[c], o);
      amr[c] += __shfl_xor_sync(0xffffffffu, amr[c], o);
      ami[c] += __shfl_xor_sync(0xffffffffu, ami[c], o);
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int c = 0; c < 7; ++c) {
      part[warp * 28 + c] = apr[c];
      part[warp * 28 + 7 + c] = api[c];
      part[warp * 28 + 14 + c] = amr[c];
      part[warp * 28 + 21 + c] = ami[c];
    }
  }
  __syncthreads();
  if (!active || half != 0 || lane >= 7) return;
  cplx *T = batch_ptr(table, cell, 0);
  const int c = lane;
  const double *pa = part + warp * 28, *pb = part + (warp + 1) * 28;  // the two halves, always summed in this order
  {
    const double sr = pa[c] + pb[c], si = pa[7 + c] + pb[7 + c];
    const int flat = (D1 + 2 * Mt) * L + D2 + 2 * Mt;
    if (origin) {
      T[(size_t)c * L2 + flat] = cmake(sr, 0.0);
    } else {
      const double inv = 1.0 / (qxp * qxp + qyp * qyp);
      const double re = si * inv, im = -sr * inv;  // (-i) (sr + i si) / |q|^2
      T[(size_t)c * L2 + flat] = cmake(re, im);
      T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(re, -im);  // T(-D) = conj T(D): Phi, R exactly Hermitian
    }
  }
  if (minus) {
    const double sr = pa[14 + c] + pb[14 + c], si = pa[21 + c] + pb[21 + c];
    const int flat = (D1 + 2 * Mt) * L - D2 + 2 * Mt;
    const double inv = 1.0 / (qxm * qxm + qym * qym);
    const double re = si * inv, im = -sr * inv;
    T[(size_t)c * L2 + flat] = cmake(re, im);
    T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(re, -im);
  }
}

int launch_table(const Geometry *geo_dev, int ncells, int Mt, BatchRef table, double total_edges, int centroid_rule,
                  cudaStream_t s, int maxP, int max_nes, BatchRef scratch, long long scratch_elems) {
  const int L = 4 * Mt + 1;
  const int nhalf = (L * L + 1) / 2;
  // algorithmic work: 118 real flops per (index difference, edge) term = the formula evaluated directly (sincospi + sinpi
  // + the division + the 7-channel accumulation), counted from the SASS of table_tma_kernel's edge loop: 50 DFMA,
  // 15 DMUL, 3 DADD (profiles/r2_s1_table.md; SURVEY 8(d) estimated ~120).  Earlier rounds used 230, which was wrong.
  KScope ks(KC_TABLE, 118.0 * total_edges * nhalf, s);
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (!centroid_rule && table_sep_smem(maxP) <= 200 * 1024 && (long long)4 * L * max_nes <= scratch_elems) {
    static unsigned long long mask = 0;
    ensure_dyn_smem(table_sep_kernel, 200 * 1024, mask);
    edge_phasor_kernel<<<dim3((max_nes + 127) / 128, L, ncells), 128, 0, s>>>(geo_dev, Mt, scratch);
    // tile TA x TB of PAIRS (D1, +-D2), D1, D2 in [0, 2Mt], per CTA (one CTA per SM), two warps per pair: the shortest
    // sequence of waves, then the most reuse of table rows
    const int n1 = 2 * Mt + 1;
    int TA = 1, TB = 1;
    long long best = -1;
    for (int a = 1; a <= 4; ++a)
      for (int b = 1; 2 * a * b <= DPB; ++b) {
        const long long tiles = (long long)((n1 + a - 1) / a) * ((n1 + b - 1) / b) * ncells;
        // a CTA's time: its warps share the FP64 pipe, but below ~8 warps the loop is bound by its own latency
        const long long cost = ((tiles + sms - 1) / sms) * (2 * a * b > 8 ? 2 * a * b : 8) * 1000 + (100 * (a + b)) / (a * b);
        if (best < 0 || cost < best) { best = cost; TA = a; TB = b; }
      }
    table_sep_kernel<<<dim3(((n1 + TA - 1) / TA) * ((n1 + TB - 1) / TB), ncells), 2 * TA * TB * 32, table_sep_smem(maxP), s>>>(
        geo_dev, Mt, table, scratch, TA, TB);
    return 2;
  }
  const size_t smem = table_tma_smem(maxP);
  if (!centroid_rule && smem <= 200 * 1024) {  // geometry and properties staged in shared memory by bulk TMA copies
    static unsigned long long mask = 0;
    ensure_dyn_smem(table_tma_kernel, 200 * 1024, mask);
    // one CTA per SM (its shared memory holds the cell's properties): as many warps per CTA as it takes to give every SM
    // one CTA, so that a single cell with few index differences still uses the whole device
    int dpb = (int)(((long long)nhalf * ncells + sms - 1) / sms);
    dpb = dpb < 1 ? 1 : (dpb > DPB ? DPB : dpb);
    table_tma_kernel<<<dim3((nhalf + dpb - 1) / dpb, ncells), dpb * 32, smem, s>>>(geo_dev, Mt, table);
    return 1;
  }
  dim3 grid(nhalf, ncells);
  table_kernel<<<grid, 256, 0, s>>>(geo_dev, Mt, table, centroid_rule);
  return 1;
}

// ---------------------------------------------------------------------------------------------- shared geometry (NEXT-3)
// Cells that share one geometry and differ in their properties (the optimisation-loop batch of PAPER.md:15-17, 297):
// the polygon integrals I_p(q_D) are evaluated once per geometry, one thread per (index difference, phase), into
// Iph[p + D_half * P]; a cell's table is then T_c(D) = sum_p w_{c,p} I_p(q_D), a (7 ncells x P) x (P x nhalf) product that
// runs on the DMMA GEMM, followed by the scatter into the cells' tables (with T(-D) = conj T(D)).
__global__ void __launch_bounds__(128) phase_table_kernel(Geometry g, const int *__restrict__ poff, int Mt, cplx *__restrict__ Iph,
                                                          int centroid_rule) {
  const int L = 4 * Mt + 1, L2 = L * L, nhalf = (L2 + 1) / 2;
  const int p = blockIdx.x * blockDim.x + threadIdx.x, dh = blockIdx.y;
  if (p >= g.P || dh >= nhalf) return;
  const int flat = dh + (L2 - 1) / 2;
  const int D1 = flat / L - 2 * Mt, D2 = flat % L - 2 * Mt;
  cplx out;
  if (D1 == 0 && D2 == 0) {
    out = cmake(g.area[p], 0.0);
  } else if (centroid_rule) {
    const double phi = fma((double)D1, g.area[g.P + p], (double)D2 * g.area[2 * g.P + p]);
    double sn, cs;
    sincospi(2.0 * phi, &sn, &cs);
    out = cmake(g.area[p] * cs, g.area[p] * sn);
  } else {
    const double qx = D1 * g.Q[0] + D2 * g.Q[2], qy = D1 * g.Q[1] + D2 * g.Q[3];
    const int ne = g.nedge, nes = g.nes;
    const double *mh1 = g.edge, *mh2 = g.edge + nes, *eh1 = g.edge + 2 * nes, *eh2 = g.edge + 3 * nes;
    const double *ex = g.edge + 4 * nes, *ey = g.edge + 5 * nes;
    double sr = 0.0, si = 0.0;
    for (int e = poff[p]; e < poff[p + 1]; ++e) {
      const double phi = fma((double)D1, mh1[e], (double)D2 * mh2[e]);  // q.m / (2 pi)
      const double u = fma((double)D1, eh1[e], (double)D2 * eh2[e]);    // q.e / (2 pi)
      double sn, cs;
      sincospi(2.0 * phi, &sn, &cs);
      const double j0 = (u == 0.0) ? 1.0 : sinpi(u) / (kPi * u);
      const double f = (qx * ey[e] - qy * ex[e]) * j0;
      sr = fma(f, cs, sr);
      si = fma(f, sn, si);
    }
    const double inv = 1.0 / (qx * qx + qy * qy);
    out = cmake(si * inv, -sr * inv);  // (-i) (sr + i si) / |q|^2
  }
  Iph[(size_t)dh * g.P + p] = out;
}

// W[(cell * 7 + c) + p * ldw] = (w_{c,p} of cell, 0): the weights of every cell of the batch as one complex matrix
__global__ void __launch_bounds__(256) gather_weights_kernel(const Geometry *__restrict__ geos, int ncells, cplx *__restrict__ W) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x, cell = blockIdx.y;
  const Geometry g = geos[cell];
  if (p >= g.P) return;
  const size_t ldw = (size_t)7 * ncells;
#pragma unroll
  for (int c = 0; c < 7; ++c) W[(size_t)cell * 7 + c + (size_t)p * ldw] = cmake(g.w[c * g.P + p], 0.0);
}

// table[c][flat] of every cell from Tst[(cell * 7 + c) + dh * ldt]; the mirrored half is the conjugate
__global__ void __launch_bounds__(256) scatter_table_kernel(int Mt, int ncells, const cplx *__restrict__ Tst, BatchRef table) {
  const int L = 4 * Mt + 1, L2 = L * L, nhalf = (L2 + 1) / 2;
  const int dh = blockIdx.x * blockDim.x + threadIdx.x, cell = blockIdx.y;
  if (dh >= nhalf) return;
  const int flat = dh + (L2 - 1) / 2;
  cplx *T = batch_ptr(table, cell, 0);
  const size_t ldt = (size_t)7 * ncells;
#pragma unroll
  for (int c = 0; c < 7; ++c) {
    cplx v = Tst[(size_t)cell * 7 + c + (size_t)dh * ldt];
    if (dh == 0) v.y = 0.0;
    T[(size_t)c * L2 + flat] = v;
    T[(size_t)c * L2 + (L2 - 1 - flat)] = cmake(v.x, -v.y);
  }
}

void launch_phase_table(const Geometry &g, const int *poff, int Mt, cplx *Iph, int centroid_rule, cudaStream_t s) {
  const int L = 4 * Mt + 1, nhalf = (L * L + 1) / 2;
  KScope ks(KC_TABLE, 118.0 * g.nedge * (double)nhalf, s);
  phase_table_kernel<<<dim3((g.P + 127) / 128, nhalf), 128, 0, s>>>(g, poff, Mt, Iph, centroid_rule);
}

void launch_shared_tables(const Geometry *geos_dev, int ncells, int P, int Mt, const cplx *Iph, cplx *W, cplx *Tst,
                          BatchRef table, cudaStream_t s) {
  const int L = 4 * Mt + 1, nhalf = (L * L + 1) / 2;
  {
    KScope ks(KC_OTHER, 0.0, s);
    gather_weights_kernel<<<dim3((P + 255) / 256, ncells), 256, 0, s>>>(geos_dev, ncells, W);
  }
  GemmDesc g{};
  g.M = 7 * ncells; g.N = nhalf; g.K = P; g.opA = 0; g.opB = 0; g.lda = 7 * ncells; g.ldb = P; g.ldc = 7 * ncells;
  g.ncells = 1; g.inner = 1; g.kclass = KC_TABLE;
  g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
  g.A = BatchRef{nullptr, (unsigned long long)W, 0, 0};
  g.B = BatchRef{nullptr, (unsigned long long)Iph, 0, 0};
  g.C = BatchRef{nullptr, (unsigned long long)Tst, 0, 0};
  launch_zgemm(g, s);
  {
    KScope ks(KC_OTHER, 0.0, s);
    scatter_table_kernel<<<dim3((nhalf + 255) / 256, ncells), 256, 0, s>>>(Mt, ncells, Tst, table);
  }
}

// S2: one thread per (g_alpha, g_beta): Phi[(a,ga),(b,gb)] = T_{c(a,b)}(D(gb) - D(ga)), R[ga,gb] = T_rho(...).
// Consecutive threads -> consecutive rows ga (column-major stores coalesce; table reads are nearly contiguous).
__global__ void __launch_bounds__(256) expand_kernel(int Mt, BatchRef table, BatchRef Phi, BatchRef R) {
  const int cell = blockIdx.z;
  const int W = 2 * Mt + 1;
  const int N = W * W;
  const int L = 4 * Mt + 1;
  const int L2 = L * L;
  const int ga = blockIdx.x * blockDim.x + threadIdx.x;
  const int gb = blockIdx.y;
  if (ga >= N) return;
  const cplx *T = batch_ptr(table, cell, 0);
  cplx *P = batch_ptr(Phi, cell, 0);
  cplx *Rm = batch_ptr(R, cell, 0);
  const int d1 = gb / W - ga / W + 2 * Mt;
  const int d2 = gb % W - ga % W + 2 * Mt;
  const int f = d1 * L + d2;
  const size_t n3 = 3 * (size_t)N;
  // channel of block (a,b): 11 22 12 13 23 33 -> 0 1 2 3 4 5
  const int chan[3][3] = {{0, 2, 3}, {2, 1, 4}, {3, 4, 5}};
#pragma unroll
  for (int b = 0; b < 3; ++b)
#pragma unroll
    for (int a = 0; a < 3; ++a) P[((size_t)b * N + gb) * n3 + (size_t)a * N + ga] = T[(size_t)chan[a][b] * L2 + f];
  Rm[(size_t)gb * N + ga] = T[(size_t)6 * L2 + f];
}

void launch_expand(int ncells, int Mt, BatchRef table, BatchRef Phi, BatchRef R, cudaStream_t s) {
  const int W = 2 * Mt + 1, N = W * W;
  dim3 grid((N + 255) / 256, N, ncells);
  KScope ks(KC_EXPAND, 160.0 * N * N * ncells, s);  // 9 + 1 blocks of N x N complex128 written once
  expand_kernel<<<grid, 256, 0, s>>>(Mt, table, Phi, R);
}

// Isotropic shortcut of S3: with Phi = [[A, B, 0], [B, A, 0], [0, 0, 2(A - B)]],
// Phi^{-1} follows from the two N x N inverses Ei = (A + B)^{-1}, Fi = (A - B)^{-1}.
// expand_sumdiff: E = A + B, F = A - B from the table channels 0 (Dv11) and 2 (Dv12).
__global__ void __launch_bounds__(256) expand_sumdiff_kernel(int Mt, BatchRef table, BatchRef E, BatchRef F) {
  const int cell = blockIdx.z;
  const int W = 2 * Mt + 1, N = W * W, L = 4 * Mt + 1, L2 = L * L;
  const int ga = blockIdx.x * blockDim.x + threadIdx.x, gb = blockIdx.y;
  if (ga >= N) return;
  const cplx *T = batch_ptr(table, cell, 0);
  const int f = (gb / W - ga / W + 2 * Mt) * L + (gb % W - ga % W + 2 * Mt);
  const cplx a = T[f], b = T[(size_t)2 * L2 + f];
  batch_ptr(E, cell, 0)[(size_t)gb * N + ga] = cadd(a, b);
  batch_ptr(F, cell, 0)[(size_t)gb * N + ga] = csub(a, b);
}
// compose: Y11 = Y22 = (Ei + Fi)/2, Y12 = Y21 = (Ei - Fi)/2, Y33 = Fi/2, all other blocks zero.
__global__ void __launch_bounds__(256) compose_y_kernel(int N, BatchRef Ei, BatchRef Fi, BatchRef Y) {
  const int cell = blockIdx.z;
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= N) return;
  const cplx e = batch_ptr(Ei, cell, 0)[(size_t)c * N + r], f = batch_ptr(Fi, cell, 0)[(size_t)c * N + r];
  cplx *Yg = batch_ptr(Y, cell, 0);
  const size_t n3 = 3 * (size_t)N;
  const cplx sum = cscale(cadd(e, f), 0.5), dif = cscale(csub(e, f), 0.5), zero = cmake(0.0, 0.0);
  const cplx blk[3][3] = {{sum, dif, zero}, {dif, sum, zero}, {zero, zero, cscale(f, 0.5)}};
#pragma unroll
  for (int b = 0; b < 3; ++b)
#pragma unroll
    for (int a = 0; a < 3; ++a) Yg[((size_t)b * N + c) * n3 + (size_t)a * N + r] = blk[a][b];
}

void launch_expand_sumdiff(int ncells, int Mt, BatchRef table, BatchRef E, BatchRef F, cudaStream_t s) {
  const int W = 2 * Mt + 1, N = W * W;
  KScope ks(KC_EXPAND, 32.0 * N * N * ncells, s);
  expand_sumdiff_kernel<<<dim3((N + 255) / 256, N, ncells), 256, 0, s>>>(Mt, table, E, F);
}
void launch_compose_y(int ncells, int N, BatchRef Ei, BatchRef Fi, BatchRef Y, cudaStream_t s) {
  KScope ks(KC_EXPAND, 16.0 * 11.0 * N * N * ncells, s);
  compose_y_kernel<<<dim3((N + 255) / 256, N, ncells), 256, 0, s>>>(N, Ei, Fi, Y);
}

}  // namespace bsk
