// C-ABI of libbs.so (include/bs.h): handle, workspace layout and the host-side orchestration of S0..S8.
// Every arithmetic step of the path runs in the kernels of assemble.cu / factor.cu / zgemm.cu / pencil.cu / tridiag.cu /
// sturm.cu; the host only does S0 (geometry preparation) and argument marshalling.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <unordered_map>

#include "bs_internal.cuh"

namespace bsk {
thread_local KTimer *g_kt = nullptr;
}

namespace {

thread_local char g_err[512] = "";

bs_status fail(bs_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}

#define CU(expr)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (expr);                                                                       \
    if (e_ != cudaSuccess) return fail(BS_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));      \
  } while (0)

constexpr double kTwoPi = 6.283185307179586476925286766559;

// Offsets (complex128 elements, each region 256-byte aligned) inside one cell's workspace.
struct Layout {
  int Mt = -1, N = 0, nk = 0, mode = 0, nb = 0;
  long long table, Phi, R, Lf, X, tmp, dinv, Y, LR, XR, tmpR, dinvR, kvecA, Coef, Tb, kvecK, Kk, Ak, VW, P, SM, AB;
  long long vw_stride, sm_stride, ab_stride;
  // mode shapes (BS_OPT_MODES = nvmax > 0): kept reflectors of stage 1, a copy of the band, vectors and scratch
  int nvmax = 0;
  long long Vall, Tall, AB2, Zv, LU, Uv, HU, Sv, Wa, Wb, kapm;
  long long lu_stride;
  long long total;  // elements
};

long long align16(long long x) { return (x + 15) & ~15LL; }
int band_width(int nb) { return nb >= 32 ? 32 : (nb >= 16 ? 16 : 8); }  // two-stage band width from BS_OPT_PANEL
// BS_OPT_PANEL = 0 (default): band width 16 for every n above the shared-memory one-stage kernel.  Measured with the
// register-tile chasing kernel of chase.cu (S6 total, ms, band width 8 / 16 / 32): n = 242 x 2000: 36.4 / 30.1 / 52.8;
// n = 338 x 1000: 37.4 / 29.6 / 47.7; n = 450 x 60: 9.9 / 7.6 / 9.1; n = 882 x 90: 45.7 / 30.7 / 33.9; n = 1300 x 100:
// - / 78.7 / 84.4; n = 1922 x 120: - / 246.1 / 250.6 (stage 2 alone 50.5 vs 85.6 ms; the narrower panels cost stage 1
// that much again at this size).  The choice does not depend on the batch, so a batch and its members take the same path.
int auto_band_width(int n) { (void)n; return 16; }

Layout make_layout(int Mt, int nk, int mode, int nb_opt, int nvmax = 0) {
  const int nb = nb_opt > 0 ? nb_opt : 32;  // automatic band width: sized for the widest
  Layout L;
  L.Mt = Mt; L.nk = nk; L.mode = mode; L.nb = nb_opt; L.nvmax = nvmax;
  const long long W = 2 * Mt + 1, N = W * W, n3 = 3 * N, n2 = 2 * N, Lt = 4 * Mt + 1;
  L.N = (int)N;
  long long o = 0;
  auto take = [&](long long elems) { long long at = o; o = align16(o + elems); return at; };
  L.table = take(7 * Lt * Lt);
  L.Phi = take(n3 * n3);
  L.R = take(N * N);
  L.Lf = take(n3 * n3);
  L.X = take(n3 * n3);
  L.tmp = take(n3 * n3);
  L.dinv = take(((n3 + 63) / 64) * 4096 + ((N + 63) / 64) * 4096);  // + a second N-sized slot (isotropic shortcut)
  L.Y = take(n3 * n3);
  L.LR = take(N * N);
  L.XR = take(N * N);
  L.tmpR = take(N * N);
  L.dinvR = take(((N + 63) / 64) * 4096);
  L.kvecA = take(6 * 2 * 2 * N);      // 6 matrices x 2 terms x [2][2][N] doubles
  L.Coef = take(mode == BS_PENCIL_POLY ? 6 * n2 * n2 : 0);
  L.Tb = take((mode == BS_PENCIL_POLY ? 6 : (long long)nk) * N * N);
  L.kvecK = take((long long)nk * 2 * N);  // nk x [2][2][N] doubles
  L.Kk = take(mode == BS_PENCIL_DIRECT ? (long long)nk * n2 * n2 : n2 * n2);  // POLY keeps one slot for bs_get_pencil
  L.Ak = take((long long)nk * n2 * n2);
  const int bw = band_width(nb);
  L.vw_stride = (long long)std::max(bsk::tridiag_vw_elems((int)n2, nb), bsk::band_vw_elems((int)n2, bw));
  L.sm_stride = align16((long long)bsk::band_sm_elems(bw));
  L.ab_stride = align16((long long)bsk::band_ab_elems((int)n2, bw));
  L.VW = take((long long)nk * L.vw_stride);
  L.P = take((long long)nk * (long long)bsk::tridiag_p_elems((int)n2));
  L.SM = take((long long)nk * L.sm_stride);
  L.AB = take((long long)nk * L.ab_stride);
  if (nvmax > 0) {
    L.Vall = take((long long)nk * n2 * n2);
    L.Tall = take((long long)nk * n2 * 32);           // (n / b) panels of b^2 <= n * 32
    L.AB2 = take((long long)nk * L.ab_stride);
    L.Zv = take((long long)nk * n2 * nvmax);
    L.lu_stride = align16((long long)bsk::band_invit_lu_elems((int)n2, 32));
    L.LU = take((long long)nk * L.lu_stride);
    L.Uv = take((long long)nk * n2 * nvmax);
    L.HU = take((long long)nk * n3 * nvmax);
    L.Sv = take((long long)nk * n3 * nvmax);
    L.Wa = take((long long)nk * 32 * nvmax);
    L.Wb = take((long long)nk * 32 * nvmax);
    L.kapm = take((long long)nk * N);                 // nk x [2][N] doubles
  }
  L.total = o;
  return L;
}

}  // namespace

// Geometry shared by the handles of bs_create_cells_shared (refcounted): edge arrays once, and the table of polygon
// integrals I_p(q_D) of the last truncation / quadrature it was assembled with.
struct SharedGeom {
  int refs = 0, device = 0, P = 0, nedge = 0;
  char *d_blob = nullptr;
  double *d_edge = nullptr, *d_area = nullptr;
  int *d_ephase = nullptr, *d_poff = nullptr;
  cplx *d_phase = nullptr;   // [P x nhalf]
  size_t phase_cap = 0;      // elements
  int phase_Mt = -1, phase_quad = -1;
};

struct bs_cell {
  double A[4], T[4], Q[4], V;
  int P = 0, nedge = 0;
  bool isotropic = true;  // every phase has the isotropic plane-strain block structure of PAPER.md:173
  int phi_general = 0;    // BS_OPT_PHI_INVERSE: 1 = always the general 3N x 3N inverse
  int out_root = 0;       // BS_OPT_OUTPUT: 1 = bs_bands writes omega = sqrt(max(lambda, 0)) instead of lambda
  char *d_blob = nullptr;  // the one device allocation that holds geo, edge, w, area, ephase
  double *d_edge = nullptr, *d_w = nullptr, *d_area = nullptr;
  int *d_ephase = nullptr;
  bsk::Geometry geo;
  bsk::Geometry *d_geo = nullptr;  // [1]
  int mode = BS_PENCIL_POLY, nb = 0, timing = 0, algo = BS_TRIDIAG_TWO_STAGE, quad = BS_ASSEMBLY_EXACT;
  void *ws = nullptr;
  size_t ws_bytes = 0;
  Layout lay;            // layout of the last bs_assemble (lay.Mt < 0: not assembled)
  int ws_nk = 0;         // nk the caller sized the workspace for (unknown: derived from bytes at assemble time)
  bool assembled = false;
  int64_t launches = 0;
  double ms[BS_T_COUNT] = {0};
  // batch scratch owned by the handle that leads a call (cells[0])
  unsigned long long *d_bases = nullptr;
  bsk::Geometry *d_geos = nullptr;
  int *d_info = nullptr;              // [5 ncells]: Phi, R, then (E, F, R) of the batched isotropic factorisation
  unsigned long long *d_bases3 = nullptr;  // [4][3 ncells] matrix addresses of that batched call
  int batch_cap = 0;
  double *d_flat = nullptr;  // d, e, scal, lam, coefk
  size_t flat_cap = 0;
  int last_n = 0, last_nmat = 0, last_nk = 0;
  cudaEvent_t ev[BS_T_COUNT + 1] = {nullptr};
  bsk::KTimer *kt = nullptr;  // BS_OPT_TIMING = 2
  int nvmax = 0;                  // BS_OPT_MODES: bs_modes may return up to this many mode shapes per k-point
  int refine = 0;                 // BS_OPT_REFINE: bs_modes returns the factored Rayleigh quotients of its modes
  bool keep_modes = false;        // set by bs_modes around its bs_bands pass: stage 1 keeps its reflectors and the band
  double *last_lam = nullptr;     // device eigenvalues of the last bs_bands pass (nmat x nbands)
  SharedGeom *shared = nullptr;   // bs_create_cells_shared
  cplx *d_sh = nullptr;           // lead handle: weights matrix and stacked tables of the shared-geometry S1
  size_t sh_cap = 0;
  // the stream of the last call that launched work reading this handle's blocks (bs_assemble / bs_bands / accessors):
  // the accessors and bs_destroy_cell wait for THAT stream only, never for the whole device
  cudaStream_t last_stream = nullptr;
  bool used = false;
  int device = 0;  // the device the handle's blocks live on (current device at bs_create_cell)
};

namespace {

BatchRef ref(const bs_cell *lead, int ncells, bs_cell *const *cells, long long off, long long stride) {
  BatchRef r;
  r.bases = ncells > 1 ? lead->d_bases : nullptr;
  r.single = (unsigned long long)cells[0]->ws;
  r.off = off;
  r.stride = stride;
  return r;
}

// Handle-owned device blocks (geometry blob, batch tables) come from a process-wide cache of freed blocks: creating and
// destroying handles in a loop (an optimisation driver, bench.py's end-to-end arm) then costs no cudaMalloc / cudaFree,
// whose latency on a busy device is erratic (measured: bs_destroy_cell 1 ms typically, 10-530 ms in one call of five).
// A block is reused only on its own device and by exact (256-byte rounded) size; at most 256 MiB stay cached.  bs_destroy_cell synchronises the
// device before it returns blocks, so a reused block has no reader left.
struct DevCache {
  std::mutex mu;
  std::multimap<std::pair<int, size_t>, void *> free_blocks;  // (device, bytes) -> block
  std::unordered_map<void *, std::pair<int, size_t>> sizes;
  size_t cached = 0;
  static size_t round(size_t b) { return (b + 255) & ~(size_t)255; }
  cudaError_t alloc(void **p, size_t bytes) {
    const size_t r = round(bytes ? bytes : 1);
    int dev = 0;
    cudaGetDevice(&dev);
    {
      std::lock_guard<std::mutex> g(mu);
      auto it = free_blocks.find({dev, r});
      if (it != free_blocks.end()) {
        *p = it->second;
        free_blocks.erase(it);
        cached -= r;
        return cudaSuccess;
      }
    }
    cudaError_t e = cudaMalloc(p, r);
    if (e == cudaSuccess) {
      std::lock_guard<std::mutex> g(mu);
      sizes[*p] = {dev, r};
    }
    return e;
  }
  void release(void *p) {  // the caller has made sure that no kernel still uses p
    if (!p) return;
    std::lock_guard<std::mutex> g(mu);
    auto it = sizes.find(p);
    if (it == sizes.end()) { cudaFree(p); return; }
    if (cached + it->second.second > ((size_t)256 << 20)) { sizes.erase(it); cudaFree(p); return; }
    free_blocks.emplace(it->second, p);
    cached += it->second.second;
  }
};
DevCache &dev_cache() { static DevCache c; return c; }
template <class T>
cudaError_t dev_alloc(T **p, size_t bytes) { return dev_cache().alloc(reinterpret_cast<void **>(p), bytes); }

// Waits for the work the handle's last call enqueued (its own stream), not for the device.
void sync_handle(const bs_cell *c) {
  if (c->used && cudaStreamSynchronize(c->last_stream) != cudaSuccess) cudaGetLastError();  // (a destroyed stream: nothing left to wait for)
}
void mark_stream(bs_cell *const *cells, int ncells, cudaStream_t s) {
  for (int c = 0; c < ncells; ++c) {
    if (cells[c]->used && cells[c]->last_stream != s) sync_handle(cells[c]);  // a handle moved to another stream: drain the old one
    cells[c]->last_stream = s;
    cells[c]->used = true;
  }
}

bs_status ensure_batch(bs_cell *lead, bs_cell *const *cells, int ncells, cudaStream_t s) {
  if (ncells > lead->batch_cap) {
    if (lead->d_bases) sync_handle(lead);  // earlier launches (on the handle's stream) may still read the tables
    dev_cache().release(lead->d_bases); dev_cache().release(lead->d_geos);
    dev_cache().release(lead->d_info); dev_cache().release(lead->d_bases3);
    lead->d_bases = nullptr; lead->d_geos = nullptr; lead->d_info = nullptr; lead->d_bases3 = nullptr; lead->batch_cap = 0;
    CU(dev_alloc(&lead->d_bases, sizeof(unsigned long long) * ncells));
    CU(dev_alloc(&lead->d_geos, sizeof(bsk::Geometry) * ncells));
    CU(dev_alloc(&lead->d_info, sizeof(int) * 5 * ncells));
    CU(dev_alloc(&lead->d_bases3, sizeof(unsigned long long) * 12 * ncells));
    lead->batch_cap = ncells;
  }
  std::vector<unsigned long long> b(ncells);
  std::vector<bsk::Geometry> g(ncells);
  for (int c = 0; c < ncells; ++c) {
    b[c] = (unsigned long long)cells[c]->ws;
    g[c] = cells[c]->geo;
  }
  CU(cudaMemcpyAsync(lead->d_bases, b.data(), sizeof(unsigned long long) * ncells, cudaMemcpyHostToDevice, s));
  CU(cudaMemcpyAsync(lead->d_geos, g.data(), sizeof(bsk::Geometry) * ncells, cudaMemcpyHostToDevice, s));
  // (no stream synchronise: an H2D copy from pageable memory is staged before cudaMemcpyAsync returns)
  return BS_OK;
}

bs_status ensure_flat(bs_cell *lead, size_t doubles) {
  if (doubles > lead->flat_cap) {
    if (lead->d_flat) { sync_handle(lead); dev_cache().release(lead->d_flat); }
    lead->d_flat = nullptr; lead->flat_cap = 0;
    CU(dev_alloc(&lead->d_flat, doubles * sizeof(double)));
    lead->flat_cap = doubles;
  }
  return BS_OK;
}

void tick(bs_cell *c, int idx, cudaStream_t s) {
  if (!c->timing) return;
  if (!c->ev[idx]) cudaEventCreate(&c->ev[idx]);
  cudaEventRecord(c->ev[idx], s);
}
struct KtGuard {  // routes the launchers' KScope to the lead cell's timer for the duration of one call
  explicit KtGuard(bs_cell *c) { bsk::g_kt = (c->timing == 2) ? c->kt : nullptr; if (bsk::g_kt) bsk::g_kt->reset(); }
  ~KtGuard() { bsk::g_kt = nullptr; }
};

// S0 on the host (PAPER.md:23-26 eq. 1, :138): reciprocal basis, fractional coordinates, per-edge arrays, signed areas and
// centroids, tiling check.
struct HostGeom {
  double T[4], Q[4], V = 0.0;
  int ne = 0, nes = 0;
  std::vector<double> edge, area;  // edge: SoA [6][ne]; area: [area | ch1 | ch2][P]
  std::vector<int> eph;
};
bs_status host_geometry(const double lattice[4], int nphase, const int32_t *vert_offset, const double *verts, HostGeom &g) {
  if (vert_offset[0] != 0) return fail(BS_ERR_ARG, "bs_create_cell: vert_offset[0] != 0");
  for (int p = 0; p < nphase; ++p)
    if (vert_offset[p + 1] - vert_offset[p] < 3) return fail(BS_ERR_ARG, "bs_create_cell: phase %d has < 3 vertices", p);
  const double det = lattice[0] * lattice[3] - lattice[1] * lattice[2];
  if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return fail(BS_ERR_GEOMETRY, "bs_create_cell: singular lattice");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(BS_ERR_CUDA, "bs_create_cell: no CUDA device");
  // T = A^{-1}; q^j = 2 pi (column j of T)  =>  q^i . h^j = 2 pi delta_ij   (PAPER.md:23-26 eq. 1, :138)
  g.T[0] = lattice[3] / det;  g.T[1] = -lattice[1] / det;
  g.T[2] = -lattice[2] / det; g.T[3] = lattice[0] / det;
  g.Q[0] = kTwoPi * g.T[0]; g.Q[1] = kTwoPi * g.T[2];  // q^1
  g.Q[2] = kTwoPi * g.T[1]; g.Q[3] = kTwoPi * g.T[3];  // q^2
  g.V = std::fabs(det);
  const int ne = vert_offset[nphase], nes = (ne + 1) & ~1;  // (SoA stride: even, so that every array is 16-byte aligned)
  g.ne = ne;
  g.nes = nes;
  g.edge.assign((size_t)6 * nes, 0.0);
  g.area.assign((size_t)3 * nphase, 0.0);
  g.eph.assign(ne, 0);
  double total = 0.0;
  for (int p = 0; p < nphase; ++p) {
    const int s = vert_offset[p], t = vert_offset[p + 1];
    double a2 = 0.0, cxs = 0.0, cys = 0.0;
    for (int i = s; i < t; ++i) {
      const int k = (i + 1 < t) ? i + 1 : s;
      const double x0 = verts[2 * i], y0 = verts[2 * i + 1], x1 = verts[2 * k], y1 = verts[2 * k + 1];
      a2 += x0 * y1 - x1 * y0;
      cxs += (x0 + x1) * (x0 * y1 - x1 * y0);
      cys += (y0 + y1) * (x0 * y1 - x1 * y0);
      const double ex = x1 - x0, ey = y1 - y0, mx = 0.5 * (x0 + x1), my = 0.5 * (y0 + y1);
      // fractional coordinates H = x T  (x = H_1 h^1 + H_2 h^2)
      g.edge[0 * (size_t)nes + i] = mx * g.T[0] + my * g.T[2];
      g.edge[1 * (size_t)nes + i] = mx * g.T[1] + my * g.T[3];
      g.edge[2 * (size_t)nes + i] = ex * g.T[0] + ey * g.T[2];
      g.edge[3 * (size_t)nes + i] = ex * g.T[1] + ey * g.T[3];
      g.edge[4 * (size_t)nes + i] = ex;
      g.edge[5 * (size_t)nes + i] = ey;
      g.eph[i] = p;
    }
    g.area[p] = 0.5 * a2;
    if (!(g.area[p] > 0.0))
      return fail(BS_ERR_GEOMETRY, "bs_create_cell: phase %d has non-positive signed area %g (must be CCW)", p, g.area[p]);
    total += g.area[p];
    // area centroid (used by the centroid-rule assembly mode, eq. 12), in fractional coordinates
    const double cx = cxs / (3.0 * a2), cy = cys / (3.0 * a2);
    g.area[(size_t)nphase + p] = cx * g.T[0] + cy * g.T[2];
    g.area[(size_t)2 * nphase + p] = cx * g.T[1] + cy * g.T[3];
  }
  if (std::fabs(total - g.V) > 1e-10 * g.V)
    return fail(BS_ERR_GEOMETRY, "bs_create_cell: phases cover area %.17g, cell area is %.17g", total, g.V);
  return BS_OK;
}
// Channel weights [7][P]: Voigt compliance with the factors 1/2/4 of PAPER.md:167-171 (eq. 20), then rho.
bs_status host_weights(int nphase, const double *compliance, const double *density, std::vector<double> &w, bool &iso) {
  w.assign((size_t)7 * nphase, 0.0);
  iso = true;
  for (int p = 0; p < nphase; ++p) {
    if (!(density[p] > 0.0)) return fail(BS_ERR_ARG, "bs_create_cell: phase %d has density <= 0", p);
    const double *D = compliance + 6 * (size_t)p;
    if (D[3] != 0.0 || D[4] != 0.0 || D[0] != D[1] || std::fabs(4.0 * D[5] - 2.0 * (D[0] - D[2])) > 1e-14 * std::fabs(D[0]))
      iso = false;
    w[0 * (size_t)nphase + p] = D[0];
    w[1 * (size_t)nphase + p] = D[1];
    w[2 * (size_t)nphase + p] = D[2];
    w[3 * (size_t)nphase + p] = 2.0 * D[3];
    w[4 * (size_t)nphase + p] = 2.0 * D[4];
    w[5 * (size_t)nphase + p] = 4.0 * D[5];
    w[6 * (size_t)nphase + p] = density[p];
  }
  return BS_OK;
}
void init_cell_host(bs_cell *c, const double lattice[4], const HostGeom &g, int nphase, bool iso) {
  std::memcpy(c->A, lattice, sizeof(double) * 4);
  std::memcpy(c->T, g.T, sizeof(double) * 4);
  std::memcpy(c->Q, g.Q, sizeof(double) * 4);
  c->V = g.V;
  c->P = nphase;
  c->nedge = g.ne;
  c->isotropic = iso;
  c->geo.nedge = g.ne; c->geo.nes = g.nes; c->geo.P = nphase;
  std::memcpy(c->geo.Q, g.Q, sizeof(double) * 4);
}

double tock(bs_cell *c, int a, int b) {
  float ms = 0.f;
  if (c->ev[a] && c->ev[b]) cudaEventElapsedTime(&ms, c->ev[a], c->ev[b]);
  return ms;
}

}  // namespace

extern "C" {

const char *bs_last_error(void) { return g_err; }

bs_status bs_isotropic_plane_strain(int32_t n, const double *E, const double *nu, double *out) {
  if (n < 0 || (n > 0 && (!E || !nu || !out))) return fail(BS_ERR_ARG, "bs_isotropic_plane_strain: null pointer or n < 0");
  for (int i = 0; i < n; ++i) {
    if (!(E[i] > 0.0) || !(nu[i] < 0.5) || !(nu[i] > -1.0))
      return fail(BS_ERR_ARG, "bs_isotropic_plane_strain: phase %d has E <= 0 or nu outside (-1, 0.5)", i);
    // PAPER.md:121 (eq. 14): D_jkmn = (1/2mu) [ (d_jm d_kn + d_jn d_km)/2 - lam/(2(mu+lam)) d_jk d_mn ]
    const double mu = E[i] / (2.0 * (1.0 + nu[i]));
    const double lam = E[i] * nu[i] / ((1.0 + nu[i]) * (1.0 - 2.0 * nu[i]));
    const double c = lam / (2.0 * (mu + lam)), h = 1.0 / (2.0 * mu);
    double *o = out + 6 * (size_t)i;
    o[0] = h * (1.0 - c);  // D1111
    o[1] = o[0];           // D2222
    o[2] = -h * c;         // D1122
    o[3] = 0.0;            // D1112
    o[4] = 0.0;            // D2212
    o[5] = 0.5 * h;        // D1212
  }
  return BS_OK;
}

bs_status bs_create_cell(const double lattice[4], int32_t nphase, const int32_t *vert_offset, const double *verts,
                         const double *compliance, const double *density, bs_cell **out) {
  if (!lattice || !vert_offset || !verts || !compliance || !density || !out || nphase < 1)
    return fail(BS_ERR_ARG, "bs_create_cell: null pointer or nphase < 1");
  *out = nullptr;
  HostGeom hg;
  bs_status st = host_geometry(lattice, nphase, vert_offset, verts, hg);
  if (st != BS_OK) return st;
  std::vector<double> w;
  bool iso = true;
  st = host_weights(nphase, compliance, density, w, iso);
  if (st != BS_OK) return st;
  bs_cell *c = new (std::nothrow) bs_cell();
  if (!c) return fail(BS_ERR_NOMEM, "bs_create_cell: host allocation failed");
  init_cell_host(c, lattice, hg, nphase, iso);
  // one device allocation and one H2D copy per cell: [Geometry | edge | w | area | ephase], each part 256-byte aligned
  auto pad = [](size_t b) { return (b + 255) & ~(size_t)255; };
  const size_t o_geo = 0, o_edge = pad(sizeof(bsk::Geometry)), o_w = o_edge + pad(sizeof(double) * hg.edge.size()),
               o_area = o_w + pad(sizeof(double) * w.size()), o_eph = o_area + pad(sizeof(double) * hg.area.size()),
               total_bytes = o_eph + pad(sizeof(int) * hg.eph.size());
  char *dev = nullptr;
  if (dev_alloc(&dev, total_bytes) != cudaSuccess) {
    delete c;
    return fail(BS_ERR_CUDA, "bs_create_cell: device allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
  }
  c->d_blob = dev;
  cudaGetDevice(&c->device);
  c->d_geo = reinterpret_cast<bsk::Geometry *>(dev + o_geo);
  c->d_edge = reinterpret_cast<double *>(dev + o_edge);
  c->d_w = reinterpret_cast<double *>(dev + o_w);
  c->d_area = reinterpret_cast<double *>(dev + o_area);
  c->d_ephase = reinterpret_cast<int *>(dev + o_eph);
  c->geo.edge = c->d_edge; c->geo.ephase = c->d_ephase; c->geo.w = c->d_w; c->geo.area = c->d_area;
  std::vector<char> host(total_bytes, 0);
  std::memcpy(host.data() + o_geo, &c->geo, sizeof(bsk::Geometry));
  std::memcpy(host.data() + o_edge, hg.edge.data(), sizeof(double) * hg.edge.size());
  std::memcpy(host.data() + o_w, w.data(), sizeof(double) * w.size());
  std::memcpy(host.data() + o_area, hg.area.data(), sizeof(double) * hg.area.size());
  std::memcpy(host.data() + o_eph, hg.eph.data(), sizeof(int) * hg.eph.size());
  if (cudaMemcpy(dev, host.data(), total_bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
    st = fail(BS_ERR_CUDA, "bs_create_cell: H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
    bs_destroy_cell(c);
    return st;
  }
  *out = c;
  return BS_OK;
}

bs_status bs_create_cells_shared(const double lattice[4], int32_t nphase, const int32_t *vert_offset, const double *verts,
                                 int32_t ncells, const double *compliance, const double *density, bs_cell **out) {
  if (!lattice || !vert_offset || !verts || !compliance || !density || !out || nphase < 1 || ncells < 1)
    return fail(BS_ERR_ARG, "bs_create_cells_shared: null pointer, nphase < 1 or ncells < 1");
  for (int i = 0; i < ncells; ++i) out[i] = nullptr;
  HostGeom hg;
  bs_status st = host_geometry(lattice, nphase, vert_offset, verts, hg);
  if (st != BS_OK) return st;
  // the geometry block shared by all handles: [edge | area | ephase | phase offsets]
  auto pad = [](size_t b) { return (b + 255) & ~(size_t)255; };
  const size_t o_edge = 0, o_area = pad(sizeof(double) * hg.edge.size()), o_eph = o_area + pad(sizeof(double) * hg.area.size()),
               o_poff = o_eph + pad(sizeof(int) * hg.eph.size()), gbytes = o_poff + pad(sizeof(int) * (nphase + 1));
  SharedGeom *sg = new (std::nothrow) SharedGeom();
  if (!sg) return fail(BS_ERR_NOMEM, "bs_create_cells_shared: host allocation failed");
  if (dev_alloc(&sg->d_blob, gbytes) != cudaSuccess) {
    delete sg;
    return fail(BS_ERR_CUDA, "bs_create_cells_shared: device allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
  }
  cudaGetDevice(&sg->device);
  sg->P = nphase; sg->nedge = hg.ne;
  sg->d_edge = reinterpret_cast<double *>(sg->d_blob + o_edge);
  sg->d_area = reinterpret_cast<double *>(sg->d_blob + o_area);
  sg->d_ephase = reinterpret_cast<int *>(sg->d_blob + o_eph);
  sg->d_poff = reinterpret_cast<int *>(sg->d_blob + o_poff);
  {
    std::vector<char> host(gbytes, 0);
    std::memcpy(host.data() + o_edge, hg.edge.data(), sizeof(double) * hg.edge.size());
    std::memcpy(host.data() + o_area, hg.area.data(), sizeof(double) * hg.area.size());
    std::memcpy(host.data() + o_eph, hg.eph.data(), sizeof(int) * hg.eph.size());
    std::memcpy(host.data() + o_poff, vert_offset, sizeof(int) * (nphase + 1));
    if (cudaMemcpy(sg->d_blob, host.data(), gbytes, cudaMemcpyHostToDevice) != cudaSuccess) {
      dev_cache().release(sg->d_blob);
      delete sg;
      return fail(BS_ERR_CUDA, "bs_create_cells_shared: H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
  }
  // per handle: [Geometry | w]; all of them in one staging buffer and one H2D copy per handle block
  const size_t o_w = pad(sizeof(bsk::Geometry)), cbytes = o_w + pad(sizeof(double) * 7 * nphase);
  std::vector<double> w;
  std::vector<char> host(cbytes, 0);
  for (int i = 0; i < ncells; ++i) {
    bool iso = true;
    st = host_weights(nphase, compliance + (size_t)i * 6 * nphase, density + (size_t)i * nphase, w, iso);
    bs_cell *c = st == BS_OK ? new (std::nothrow) bs_cell() : nullptr;
    if (st == BS_OK && !c) st = fail(BS_ERR_NOMEM, "bs_create_cells_shared: host allocation failed");
    if (st == BS_OK) {
      init_cell_host(c, lattice, hg, nphase, iso);
      c->shared = sg;
      ++sg->refs;
      out[i] = c;
      c->device = sg->device;
      if (dev_alloc(&c->d_blob, cbytes) != cudaSuccess) st = fail(BS_ERR_CUDA, "bs_create_cells_shared: device allocation failed");
    }
    if (st == BS_OK) {
      c->d_geo = reinterpret_cast<bsk::Geometry *>(c->d_blob);
      c->d_w = reinterpret_cast<double *>(c->d_blob + o_w);
      c->d_edge = sg->d_edge; c->d_area = sg->d_area; c->d_ephase = sg->d_ephase;
      c->geo.edge = c->d_edge; c->geo.ephase = c->d_ephase; c->geo.w = c->d_w; c->geo.area = c->d_area;
      std::memcpy(host.data(), &c->geo, sizeof(bsk::Geometry));
      std::memcpy(host.data() + o_w, w.data(), sizeof(double) * w.size());
      if (cudaMemcpy(c->d_blob, host.data(), cbytes, cudaMemcpyHostToDevice) != cudaSuccess)
        st = fail(BS_ERR_CUDA, "bs_create_cells_shared: H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    if (st != BS_OK) {
      const std::string msg = g_err;
      int owners = 0;
      for (int j = 0; j <= i; ++j) owners += out[j] != nullptr;
      for (int j = 0; j <= i; ++j) {
        if (out[j]) bs_destroy_cell(out[j]);  // (the last one frees the shared geometry)
        out[j] = nullptr;
      }
      if (owners == 0) {  // no handle ever took ownership of the geometry
        dev_cache().release(sg->d_blob);
        delete sg;
      }
      std::snprintf(g_err, sizeof(g_err), "%s", msg.c_str());
      return st;
    }
  }
  return BS_OK;
}

bs_status bs_set_properties(bs_cell *c, const double *compliance, const double *density) {
  if (!c || !compliance || !density) return fail(BS_ERR_ARG, "bs_set_properties: null argument");
  std::vector<double> w;
  bool iso = true;
  bs_status st = host_weights(c->P, compliance, density, w, iso);
  if (st != BS_OK) return st;
  sync_handle(c);  // the kernels of the last call may still read the old weights
  CU(cudaMemcpy(c->d_w, w.data(), sizeof(double) * w.size(), cudaMemcpyHostToDevice));
  c->isotropic = iso;
  c->assembled = false;
  return BS_OK;
}

void bs_destroy_cell(bs_cell *c) {
  if (!c) return;
  sync_handle(c);  // nothing in flight reads the handle's blocks once this returns (only its own stream is drained)
  DevCache &dc = dev_cache();
  dc.release(c->d_blob);
  dc.release(c->d_bases); dc.release(c->d_geos); dc.release(c->d_info); dc.release(c->d_bases3); dc.release(c->d_flat);
  dc.release(c->d_sh);
  if (c->shared && --c->shared->refs == 0) {
    dc.release(c->shared->d_blob);
    dc.release(c->shared->d_phase);
    delete c->shared;
  }
  for (auto &e : c->ev)
    if (e) cudaEventDestroy(e);
  delete c->kt;
  delete c;
}

bs_status bs_set_option(bs_cell *c, int32_t option, int32_t value) {
  if (!c) return fail(BS_ERR_ARG, "bs_set_option: null handle");
  switch (option) {
    case BS_OPT_PENCIL_MODE:
      if (value != BS_PENCIL_POLY && value != BS_PENCIL_DIRECT) return fail(BS_ERR_ARG, "bs_set_option: bad pencil mode");
      if (c->mode != value) c->assembled = false;
      c->mode = value;
      return BS_OK;
    case BS_OPT_PANEL:
      if (value != 0 && (value < 4 || value > 32 || value % 4))
        return fail(BS_ERR_ARG, "bs_set_option: panel must be 0 (automatic) or 4..32, multiple of 4");
      if (c->nb != value) c->assembled = false;
      c->nb = value;
      return BS_OK;
    case BS_OPT_TRIDIAG:
      if (value != BS_TRIDIAG_TWO_STAGE && value != BS_TRIDIAG_ONE_STAGE && value != BS_TRIDIAG_TWO_STAGE_STREAMED)
        return fail(BS_ERR_ARG, "bs_set_option: bad S6 algorithm");
      c->algo = value;
      return BS_OK;
    case BS_OPT_ASSEMBLY:
      if (value != BS_ASSEMBLY_EXACT && value != BS_ASSEMBLY_CENTROID) return fail(BS_ERR_ARG, "bs_set_option: bad assembly mode");
      if (c->quad != value) c->assembled = false;
      c->quad = value;
      return BS_OK;
    case BS_OPT_PHI_INVERSE:
      if (value != 0 && value != 1) return fail(BS_ERR_ARG, "bs_set_option: bad Phi-inverse mode");
      if (c->phi_general != value) c->assembled = false;
      c->phi_general = value;
      return BS_OK;
    case BS_OPT_OUTPUT:
      if (value != BS_OUTPUT_OMEGA2 && value != BS_OUTPUT_OMEGA) return fail(BS_ERR_ARG, "bs_set_option: bad output mode");
      c->out_root = value;
      return BS_OK;
    case BS_OPT_MODES:
      if (value < 0 || value > 2048) return fail(BS_ERR_ARG, "bs_set_option: BS_OPT_MODES must be 0..2048");
      if (c->nvmax != value) c->assembled = false;
      c->nvmax = value;
      return BS_OK;
    case BS_OPT_REFINE:
      if (value != 0 && value != 1) return fail(BS_ERR_ARG, "bs_set_option: BS_OPT_REFINE must be 0 or 1");
      c->refine = value;
      return BS_OK;
    case BS_OPT_TIMING:
      if (value < 0 || value > 2) return fail(BS_ERR_ARG, "bs_set_option: timing must be 0, 1 or 2");
      c->timing = value;
      if (value == 2 && !c->kt) c->kt = new bsk::KTimer();
      return BS_OK;
  }
  return fail(BS_ERR_ARG, "bs_set_option: unknown option %d", option);
}

bs_status bs_workspace_bytes(const bs_cell *c, int32_t Mt, int32_t nk, size_t *bytes) {
  if (!c || !bytes || Mt < 0 || nk < 1) return fail(BS_ERR_ARG, "bs_workspace_bytes: bad argument");
  const long long n2 = 2LL * (2 * Mt + 1) * (2 * Mt + 1);
  if (n2 > 2048) return fail(BS_ERR_ARG, "bs_workspace_bytes: 2N = %lld exceeds 2048", n2);
  *bytes = (size_t)make_layout(Mt, nk, c->mode, c->nb, c->nvmax).total * sizeof(cplx);
  return BS_OK;
}

bs_status bs_set_workspace(bs_cell *c, void *dev_ptr, size_t bytes) {
  if (!c || !dev_ptr) return fail(BS_ERR_ARG, "bs_set_workspace: null argument");
  if (((uintptr_t)dev_ptr) & 255) return fail(BS_ERR_ARG, "bs_set_workspace: pointer not 256-byte aligned");
  c->ws = dev_ptr;
  c->ws_bytes = bytes;
  c->assembled = false;
  return BS_OK;
}

int64_t bs_launch_count(const bs_cell *c) { return c ? c->launches : 0; }

bs_status bs_get_kernel_timings(bs_cell *c, double *ms_out, double *work_out, int64_t *count_out) {
  if (!c || !ms_out || !work_out || !count_out) return fail(BS_ERR_ARG, "bs_get_kernel_timings: null argument");
  if (!c->kt) return fail(BS_ERR_STATE, "bs_get_kernel_timings: set BS_OPT_TIMING = 2 first");
  for (int i = 0; i < BS_KC_COUNT; ++i) {
    ms_out[i] = c->kt->ms[i];
    work_out[i] = c->kt->work[i];
    count_out[i] = c->kt->count[i];
  }
  return BS_OK;
}

bs_status bs_get_timings(bs_cell *c, double *ms_out) {
  if (!c || !ms_out) return fail(BS_ERR_ARG, "bs_get_timings: null argument");
  std::memcpy(ms_out, c->ms, sizeof(double) * BS_T_COUNT);
  return BS_OK;
}

}  // extern "C"

namespace {

// k-independent direction vectors of the bilinear scaling kernel for the six coefficient matrices of
//   K(k) = V^2 Bt(G + k)^T Y Bt(G + k) = C0 + kx C1 + ky C2 + kx^2 C3 + kx ky C4 + ky^2 C5     (S4)
// layout per matrix: [2 terms][L,R][x,y][N] doubles.
void fill_coef_kvec(const bs_cell *c, int Mt, std::vector<double> &kv) {
  const int W = 2 * Mt + 1, N = W * W;
  kv.assign((size_t)6 * 8 * N, 0.0);
  std::vector<double> Gx(N), Gy(N);
  for (int a1 = -Mt; a1 <= Mt; ++a1)
    for (int a2 = -Mt; a2 <= Mt; ++a2) {
      const int g = (a1 + Mt) * W + (a2 + Mt);  // PAPER.md:150 (0-based)
      Gx[g] = a1 * c->Q[0] + a2 * c->Q[2];
      Gy[g] = a1 * c->Q[1] + a2 * c->Q[3];
    }
  // vec kinds: 0 = G, 1 = ex (1,0), 2 = ey (0,1)
  const int terms[6][2][2] = {{{0, 0}, {-1, -1}}, {{0, 1}, {1, 0}}, {{0, 2}, {2, 0}},
                              {{1, 1}, {-1, -1}}, {{1, 2}, {2, 1}}, {{2, 2}, {-1, -1}}};
  for (int m = 0; m < 6; ++m)
    for (int t = 0; t < 2; ++t)
      for (int side = 0; side < 2; ++side) {
        const int kind = terms[m][t][side];
        if (kind < 0) continue;
        double *x = &kv[(((size_t)m * 2 + t) * 2 + side) * 2 * N], *y = x + N;
        for (int g = 0; g < N; ++g) {
          x[g] = kind == 0 ? Gx[g] : (kind == 1 ? 1.0 : 0.0);
          y[g] = kind == 0 ? Gy[g] : (kind == 2 ? 1.0 : 0.0);
        }
      }
}

// kappa_g = k + G_g for every k-point: [nk][L,R][x,y][N] doubles (L = R).
void fill_direct_kvec(const bs_cell *c, int Mt, int nk, const double *kpts, std::vector<double> &kv) {
  const int W = 2 * Mt + 1, N = W * W;
  kv.assign((size_t)nk * 4 * N, 0.0);
  for (int k = 0; k < nk; ++k)
    for (int a1 = -Mt; a1 <= Mt; ++a1)
      for (int a2 = -Mt; a2 <= Mt; ++a2) {
        const int g = (a1 + Mt) * W + (a2 + Mt);
        const double f1 = kpts[2 * k] + a1, f2 = kpts[2 * k + 1] + a2;  // PAPER.md:133-138 (eq. 16): Q + alpha
        const double kx = f1 * c->Q[0] + f2 * c->Q[2], ky = f1 * c->Q[1] + f2 * c->Q[3];
        double *b = &kv[(size_t)k * 4 * N];
        b[g] = kx; b[N + g] = ky; b[2 * N + g] = kx; b[3 * N + g] = ky;
      }
}

// S5 on `inner` matrices per cell: A_jl = X_R K_jl X_R^H for the blocks (0,0), (1,0), (1,1) (lower triangle of A).
int reduce_blocks(bs_cell *lead, bs_cell *const *cells, int ncells, const Layout &L, long long src_off, long long dst_off,
                  int inner, cudaStream_t s) {
  const int N = L.N, n2 = 2 * N;
  int launches = 0;
  const long long blk[3] = {0, N, (long long)N * n2 + N};
  for (int b = 0; b < 3; ++b) {
    bsk::GemmDesc g{};
    g.ncells = ncells; g.inner = inner; g.kclass = bsk::KC_GEMM_REDUCE;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    // T = X_R * K_blk      (X_R lower: op(A)[m][k] = 0 for k > m)
    g.M = N; g.N = N; g.K = N; g.opA = 0; g.opB = 0;
    g.A = ref(lead, ncells, cells, L.XR, 0); g.lda = N;
    g.B = ref(lead, ncells, cells, src_off + blk[b], (long long)n2 * n2); g.ldb = n2;
    g.C = ref(lead, ncells, cells, L.Tb, (long long)N * N); g.ldc = N;
    g.flags = BS_GEMM_KHI_ROW;
    bsk::launch_zgemm(g, s);
    // A_blk = T * X_R^H    (op(B)[k][n] = conj(X_R[n][k]) = 0 for k > n)
    g.opB = 1;
    g.A = g.C; g.lda = N;
    g.B = ref(lead, ncells, cells, L.XR, 0); g.ldb = N;
    g.C = ref(lead, ncells, cells, dst_off + blk[b], (long long)n2 * n2); g.ldc = n2;
    g.flags = BS_GEMM_KHI_COL | (b != 1 ? BS_GEMM_LOWER_ONLY : 0);
    bsk::launch_zgemm(g, s);
    launches += 2;
  }
  return launches;
}

bs_status check_batch(bs_cell *const *cells, int ncells, const char *who) {
  if (!cells || ncells < 1) return fail(BS_ERR_ARG, "%s: no cells", who);
  for (int c = 0; c < ncells; ++c) {
    if (!cells[c]) return fail(BS_ERR_ARG, "%s: cells[%d] is null", who, c);
    if (!cells[c]->ws) return fail(BS_ERR_NOMEM, "%s: cells[%d] has no workspace (bs_set_workspace)", who, c);
    if (cells[c]->mode != cells[0]->mode || cells[c]->nb != cells[0]->nb || cells[c]->algo != cells[0]->algo ||
        cells[c]->quad != cells[0]->quad || cells[c]->nvmax != cells[0]->nvmax || cells[c]->phi_general != cells[0]->phi_general || cells[c]->out_root != cells[0]->out_root)
      return fail(BS_ERR_ARG, "%s: cells[%d] has different options than cells[0]", who, c);
    // one V^2 scales K(k) of every cell of a launch (both pencil modes): the cells of a batch share the cell area
    if (cells[c]->V != cells[0]->V)
      return fail(BS_ERR_ARG, "%s: cells[%d] has cell area %.17g, cells[0] has %.17g (a batch needs equal cell areas)", who, c,
                  cells[c]->V, cells[0]->V);
    if (cells[c]->device != cells[0]->device) return fail(BS_ERR_ARG, "%s: cells[%d] lives on another device", who, c);
  }
  return BS_OK;
}

}  // namespace

extern "C" {

bs_status bs_assemble_batch(bs_cell *const *cells, int32_t ncells, int32_t Mt, void *stream) {
  bs_status st = check_batch(cells, ncells, "bs_assemble");
  if (st != BS_OK) return st;
  if (Mt < 0) return fail(BS_ERR_ARG, "bs_assemble: truncation < 0");
  const long long N = (2LL * Mt + 1) * (2 * Mt + 1);
  if (2 * N > 2048) return fail(BS_ERR_ARG, "bs_assemble: 2N = %lld exceeds 2048", 2 * N);
  bs_cell *lead = cells[0];
  cudaStream_t s = (cudaStream_t)stream;
  const Layout L = make_layout(Mt, 1, lead->mode, lead->nb, lead->nvmax);
  for (int c = 0; c < ncells; ++c) {
    cells[c]->assembled = false;
    if ((size_t)L.total * sizeof(cplx) > cells[c]->ws_bytes)
      return fail(BS_ERR_NOMEM, "bs_assemble: cells[%d] workspace is %zu bytes, need %zu", c, cells[c]->ws_bytes,
                  (size_t)L.total * sizeof(cplx));
  }
  mark_stream(cells, ncells, s);
  st = ensure_batch(lead, cells, ncells, s);
  if (st != BS_OK) return st;
  const int n3 = 3 * (int)N, n2 = 2 * (int)N, Ni = (int)N;
  auto R = [&](long long off, long long stride = 0) { return ref(lead, ncells, cells, off, stride); };
  int64_t nl = 0;
  KtGuard ktg(lead);

  tick(lead, 0, s);
  double total_edges = 0.0;
  for (int c = 0; c < ncells; ++c) total_edges += cells[c]->nedge;
  SharedGeom *sg = lead->shared;
  for (int c = 0; c < ncells; ++c)
    if (cells[c]->shared != sg) sg = nullptr;
  if (sg) {
    // S1 with one geometry for the whole batch: polygon integrals once (kept with the geometry), then T = W I per cell
    const long long Lt = 4LL * Mt + 1, nhalf = (Lt * Lt + 1) / 2;
    if (sg->phase_Mt != Mt || sg->phase_quad != lead->quad) {
      const size_t need = (size_t)nhalf * sg->P;
      if (need > sg->phase_cap) {
        sync_handle(lead);
        dev_cache().release(sg->d_phase);
        sg->d_phase = nullptr; sg->phase_cap = 0;
        CU(dev_alloc(&sg->d_phase, need * sizeof(cplx)));
        sg->phase_cap = need;
      }
      bsk::launch_phase_table(lead->geo, sg->d_poff, Mt, sg->d_phase, lead->quad, s); ++nl;
      sg->phase_Mt = Mt; sg->phase_quad = lead->quad;
    }
    const size_t wel = (size_t)7 * ncells * sg->P, tel = (size_t)7 * ncells * nhalf;
    if (wel + tel > lead->sh_cap) {
      sync_handle(lead);
      dev_cache().release(lead->d_sh);
      lead->d_sh = nullptr; lead->sh_cap = 0;
      CU(dev_alloc(&lead->d_sh, (wel + tel) * sizeof(cplx)));
      lead->sh_cap = wel + tel;
    }
    bsk::launch_shared_tables(ncells > 1 ? lead->d_geos : lead->d_geo, ncells, sg->P, Mt, sg->d_phase, lead->d_sh,
                              lead->d_sh + wel, R(L.table), s); nl += 3;
  } else {
    int maxP = 0, max_nes = 0;
    for (int c = 0; c < ncells; ++c) {
      maxP = std::max(maxP, cells[c]->P);
      max_nes = std::max(max_nes, cells[c]->geo.nes);
    }
    // S1; scratch for the separable-phase table: the regions Lf, X, tmp of the workspace (contiguous, first written by S3)
    nl += bsk::launch_table(ncells > 1 ? lead->d_geos : lead->d_geo, ncells, Mt, R(L.table), total_edges, lead->quad, s, maxP,
                            max_nes, R(L.Lf), L.dinv - L.Lf);
  }
  tick(lead, 1, s);
  bsk::launch_expand(ncells, Mt, R(L.table), R(L.Phi), R(L.R), s); ++nl;                      // S2
  tick(lead, 2, s);
  // S3: Phi = L L^H, X = L^{-1}, Y = X^H X;  R = L_R L_R^H, X_R = L_R^{-1}
  CU(cudaMemsetAsync(lead->d_info, 0, sizeof(int) * 5 * ncells, s));
  bsk::launch_copy_matrix(Ni, Ni, R(L.R), Ni, R(L.LR), Ni, ncells, 1, s); ++nl;
  bool iso = !lead->phi_general;
  for (int c = 0; c < ncells; ++c) iso = iso && cells[c]->isotropic;
  if (!iso) nl += bsk::potrf_trtri(Ni, Ni, R(L.LR), R(L.XR), R(L.tmpR), R(L.dinvR), lead->d_info + ncells, 0, ncells, 1, s);
  if (iso) {
    // isotropic phases: Phi^{-1} from (A+B)^{-1} and (A-B)^{-1}, two N x N inverses instead of one 3N x 3N
    const long long NN = (long long)Ni * Ni;
    bsk::launch_expand_sumdiff(ncells, Mt, R(L.table), R(L.Lf), R(L.Lf + NN), s); ++nl;
    {  // E, F and R (all N x N) are factored and inverted as ONE batch of 3 ncells matrices (one latency chain)
      const long long dN = (long long)((Ni + 63) / 64) * 4096;
      const long long offs[4][3] = {{L.Lf, L.Lf + NN, L.LR}, {L.X, L.X + NN, L.XR}, {L.tmp, L.tmp + NN, L.tmpR},
                                    {L.dinv, L.dinv + dN, L.dinvR}};
      std::vector<unsigned long long> hb((size_t)12 * ncells);
      for (int a4 = 0; a4 < 4; ++a4)
        for (int c = 0; c < ncells; ++c)
          for (int w = 0; w < 3; ++w)
            hb[((size_t)a4 * ncells + c) * 3 + w] = (unsigned long long)((cplx *)cells[c]->ws + offs[a4][w]);
      CU(cudaMemcpyAsync(lead->d_bases3, hb.data(), sizeof(unsigned long long) * hb.size(), cudaMemcpyHostToDevice, s));
      // (no stream synchronise: an H2D copy from pageable memory is staged before cudaMemcpyAsync returns)
      auto B3 = [&](int a4) { BatchRef r; r.bases = lead->d_bases3 + (size_t)a4 * 3 * ncells; r.single = 0; r.off = 0; r.stride = 0; return r; };
      nl += bsk::potrf_trtri(Ni, Ni, B3(0), B3(1), B3(2), B3(3), lead->d_info + 2 * ncells, 0, 3 * ncells, 1, s);
    }
    for (int w = 0; w < 2; ++w) {
      bsk::GemmDesc g{};
      g.ncells = ncells; g.inner = 1; g.kclass = bsk::KC_GEMM_FACTOR;
      g.M = Ni; g.N = Ni; g.K = Ni; g.opA = 1; g.opB = 0;
      g.A = R(L.X + w * NN); g.lda = Ni; g.B = g.A; g.ldb = Ni; g.C = R(L.tmp + (2 + w) * NN); g.ldc = Ni;
      g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
      g.flags = BS_GEMM_LOWER_ONLY | BS_GEMM_KLO_ROW | BS_GEMM_KLO_COL;
      bsk::launch_zgemm(g, s); ++nl;
      bsk::launch_hermitian_fill_upper(Ni, R(L.tmp + (2 + w) * NN), Ni, ncells, 1, s); ++nl;
    }
    bsk::launch_compose_y(ncells, Ni, R(L.tmp + 2 * NN), R(L.tmp + 3 * NN), R(L.Y), s); ++nl;
  } else {
    bsk::launch_copy_matrix(n3, n3, R(L.Phi), n3, R(L.Lf), n3, ncells, 1, s); ++nl;
    nl += bsk::potrf_trtri(n3, n3, R(L.Lf), R(L.X), R(L.tmp), R(L.dinv), lead->d_info, 0, ncells, 1, s);
    bsk::GemmDesc g{};
    g.ncells = ncells; g.inner = 1; g.kclass = bsk::KC_GEMM_FACTOR;
    g.M = n3; g.N = n3; g.K = n3; g.opA = 1; g.opB = 0;
    g.A = R(L.X); g.lda = n3; g.B = R(L.X); g.ldb = n3; g.C = R(L.Y); g.ldc = n3;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    g.flags = BS_GEMM_LOWER_ONLY | BS_GEMM_KLO_ROW | BS_GEMM_KLO_COL;
    bsk::launch_zgemm(g, s); ++nl;
    bsk::launch_hermitian_fill_upper(n3, R(L.Y), n3, ncells, 1, s); ++nl;
  }
  tick(lead, 3, s);
  if (lead->mode == BS_PENCIL_POLY) {
    std::vector<double> kv;
    for (int c = 0; c < ncells; ++c) {
      fill_coef_kvec(cells[c], Mt, kv);
      CU(cudaMemcpyAsync((cplx *)cells[c]->ws + L.kvecA, kv.data(), kv.size() * sizeof(double), cudaMemcpyHostToDevice, s));
      // (no stream synchronise: an H2D copy from pageable memory is staged before cudaMemcpyAsync returns)
    }
    // (check_batch has made sure that the cells of the batch share one cell area V)
    bsk::launch_pencil(Ni, lead->V * lead->V, R(L.Y), n3, R(L.Coef, (long long)n2 * n2), n2, R(L.kvecA, 4LL * Ni), 2,
                       ncells, 6, s); ++nl;
    nl += reduce_blocks(lead, cells, ncells, L, L.Coef, L.Coef, 6, s);
  }
  tick(lead, 4, s);
  CU(cudaStreamSynchronize(s));
  CU(cudaGetLastError());
  if (bsk::g_kt) bsk::g_kt->collect();
  std::vector<int> info(2 * ncells);
  std::vector<int> info5(5 * ncells);
  CU(cudaMemcpy(info5.data(), lead->d_info, sizeof(int) * 5 * ncells, cudaMemcpyDeviceToHost));
  for (int c = 0; c < ncells; ++c) {
    const int *b3 = &info5[2 * ncells + 3 * c];  // batched isotropic path: E, F -> Phi; R
    info[c] = info5[c] ? info5[c] : (b3[0] ? b3[0] : b3[1]);
    info[ncells + c] = info5[ncells + c] ? info5[ncells + c] : b3[2];
  }
  lead->launches += nl;
  if (lead->timing) {
    lead->ms[BS_T_TABLE] = tock(lead, 0, 1);
    lead->ms[BS_T_EXPAND] = tock(lead, 1, 2);
    lead->ms[BS_T_FACTOR] = tock(lead, 2, 3);
    lead->ms[BS_T_COEF] = tock(lead, 3, 4);
  }
  for (int c = 0; c < ncells; ++c) {
    if (info[c]) return fail(BS_ERR_NOT_PD, "bs_assemble: Phi of cells[%d] is not positive definite (pivot %d)", c, info[c]);
    if (info[ncells + c])
      return fail(BS_ERR_NOT_PD, "bs_assemble: R (Psi) of cells[%d] is not positive definite (pivot %d)", c, info[ncells + c]);
  }
  for (int c = 0; c < ncells; ++c) {
    cells[c]->lay = L;
    cells[c]->assembled = true;
  }
  return BS_OK;
}

bs_status bs_assemble(bs_cell *cell, int32_t Mt, void *stream) {
  if (!cell) return fail(BS_ERR_ARG, "bs_assemble: null handle");
  return bs_assemble_batch(&cell, 1, Mt, stream);
}

bs_status bs_get_table(bs_cell *c, void *table_host) {
  if (!c || !table_host) return fail(BS_ERR_ARG, "bs_get_table: null argument");
  if (!c->assembled) return fail(BS_ERR_STATE, "bs_get_table: call bs_assemble first");
  const long long Lt = 4 * c->lay.Mt + 1;
  sync_handle(c);
  CU(cudaMemcpy(table_host, (cplx *)c->ws + c->lay.table, sizeof(cplx) * 7 * Lt * Lt, cudaMemcpyDeviceToHost));
  return BS_OK;
}

bs_status bs_get_matrices(bs_cell *c, void *phi_host, void *psi_host) {
  if (!c) return fail(BS_ERR_ARG, "bs_get_matrices: null handle");
  if (!c->assembled) return fail(BS_ERR_STATE, "bs_get_matrices: call bs_assemble first");
  const size_t N = c->lay.N, n3 = 3 * N, n2 = 2 * N;
  sync_handle(c);
  if (phi_host) CU(cudaMemcpy(phi_host, (cplx *)c->ws + c->lay.Phi, sizeof(cplx) * n3 * n3, cudaMemcpyDeviceToHost));
  if (psi_host) {  // Psi = diag(R, R)  (eq. 19)
    std::memset(psi_host, 0, sizeof(cplx) * n2 * n2);
    const cplx *Rd = (cplx *)c->ws + c->lay.R;
    cplx *ps = (cplx *)psi_host;
    CU(cudaMemcpy2D(ps, sizeof(cplx) * n2, Rd, sizeof(cplx) * N, sizeof(cplx) * N, N, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy2D(ps + N * n2 + N, sizeof(cplx) * n2, Rd, sizeof(cplx) * N, sizeof(cplx) * N, N, cudaMemcpyDeviceToHost));
  }
  return BS_OK;
}

bs_status bs_get_pencil(bs_cell *c, const double kred[2], void *K_host, void *stream) {
  if (!c || !kred || !K_host) return fail(BS_ERR_ARG, "bs_get_pencil: null argument");
  if (!c->assembled) return fail(BS_ERR_STATE, "bs_get_pencil: call bs_assemble first");
  cudaStream_t s = (cudaStream_t)stream;
  const Layout L = make_layout(c->lay.Mt, 1, c->mode, c->nb, c->nvmax);
  const int N = L.N, n2 = 2 * N, n3 = 3 * N;
  std::vector<double> kv;
  fill_direct_kvec(c, L.Mt, 1, kred, kv);
  CU(cudaMemcpyAsync((cplx *)c->ws + L.kvecK, kv.data(), kv.size() * sizeof(double), cudaMemcpyHostToDevice, s));
  bs_cell *cells[1] = {c};
  mark_stream(cells, 1, s);
  bsk::launch_pencil(N, c->V * c->V, ref(c, 1, cells, L.Y, 0), n3, ref(c, 1, cells, L.Kk, 0), n2,
                     ref(c, 1, cells, L.kvecK, 0), 1, 1, 1, s);
  c->launches += 1;
  CU(cudaMemcpyAsync(K_host, (cplx *)c->ws + L.Kk, sizeof(cplx) * n2 * n2, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return BS_OK;
}

}  // extern "C"

extern "C" {

bs_status bs_bands_batch(bs_cell *const *cells, int32_t ncells, int32_t nk, const double *kpts, int32_t nbands,
                         double *omega2_out, void *stream) {
  bs_status st = check_batch(cells, ncells, "bs_bands");
  if (st != BS_OK) return st;
  if (!kpts || !omega2_out || nk < 1) return fail(BS_ERR_ARG, "bs_bands: null pointer or nk < 1");
  bs_cell *lead = cells[0];
  for (int c = 0; c < ncells; ++c) {
    if (!cells[c]->assembled) return fail(BS_ERR_STATE, "bs_bands: cells[%d] is not assembled (bs_assemble)", c);
    if (cells[c]->lay.Mt != lead->lay.Mt) return fail(BS_ERR_ARG, "bs_bands: cells[%d] has a different truncation", c);
  }
  const int Mt = lead->lay.Mt;
  const Layout L = make_layout(Mt, nk, lead->mode, lead->nb, lead->nvmax);
  const int N = L.N, n2 = 2 * N, n3 = 3 * N;
  if (nbands < 1 || nbands > n2) return fail(BS_ERR_ARG, "bs_bands: nbands must be in 1..2N = %d", n2);
  if ((long long)ncells * nk > 65535) return fail(BS_ERR_ARG, "bs_bands: ncells * nk = %lld exceeds 65535 matrices per call", (long long)ncells * nk);
  for (int c = 0; c < ncells; ++c)
    if ((size_t)L.total * sizeof(cplx) > cells[c]->ws_bytes)
      return fail(BS_ERR_NOMEM, "bs_bands: cells[%d] workspace is %zu bytes, %d k-points need %zu", c, cells[c]->ws_bytes, nk,
                  (size_t)L.total * sizeof(cplx));
  cudaStream_t s = (cudaStream_t)stream;
  mark_stream(cells, ncells, s);
  st = ensure_batch(lead, cells, ncells, s);
  if (st != BS_OK) return st;
  const size_t nmat = (size_t)ncells * nk;
  // flat scratch: d, e (nmat x n), scal (2 nmat), lam (nmat x nbands), coefk (6 nmat)
  const size_t nsync = bsk::sb2st_sync_ints(n2, (int)nmat);
  st = ensure_flat(lead, nmat * ((size_t)2 * n2 + 2 + nbands + 6) + (nsync + 1) / 2);
  if (st != BS_OK) return st;
  double *d = lead->d_flat, *e = d + nmat * n2, *scal = e + nmat * n2, *lam = scal + 2 * nmat, *coefk = lam + nmat * nbands;
  int *chase_sync = reinterpret_cast<int *>(coefk + 6 * nmat);
  auto R = [&](long long off, long long stride = 0) { return ref(lead, ncells, cells, off, stride); };
  int64_t nl = 0;
  KtGuard ktg(lead);
  const long long mat = (long long)n2 * n2;

  tick(lead, 0, s);
  if (lead->mode == BS_PENCIL_POLY) {
    std::vector<double> ck(nmat * 6);
    for (int c = 0; c < ncells; ++c)
      for (int k = 0; k < nk; ++k) {
        const double *Q = cells[c]->Q;
        const double kx = kpts[2 * k] * Q[0] + kpts[2 * k + 1] * Q[2], ky = kpts[2 * k] * Q[1] + kpts[2 * k + 1] * Q[3];
        double *o = &ck[((size_t)c * nk + k) * 6];
        o[0] = 1.0; o[1] = kx; o[2] = ky; o[3] = kx * kx; o[4] = kx * ky; o[5] = ky * ky;
      }
    CU(cudaMemcpyAsync(coefk, ck.data(), ck.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    // (no stream synchronise: an H2D copy from pageable memory is staged before cudaMemcpyAsync returns)
    bsk::launch_combine(n2, R(L.Coef), mat, R(L.Ak, mat), n2, coefk, nk, ncells, s); ++nl;
  } else {
    std::vector<double> kv;
    for (int c = 0; c < ncells; ++c) {
      fill_direct_kvec(cells[c], Mt, nk, kpts, kv);
      CU(cudaMemcpyAsync((cplx *)cells[c]->ws + L.kvecK, kv.data(), kv.size() * sizeof(double), cudaMemcpyHostToDevice, s));
      // (no stream synchronise: an H2D copy from pageable memory is staged before cudaMemcpyAsync returns)
    }
    bsk::launch_pencil(N, lead->V * lead->V, R(L.Y), n3, R(L.Kk, mat), n2, R(L.kvecK, 2LL * N), 1, ncells, nk, s); ++nl;  // S4
    nl += reduce_blocks(lead, cells, ncells, L, L.Kk, L.Ak, nk, s);                                                        // S5
  }
  tick(lead, 1, s);
  if (lead->keep_modes) {
    // mode shapes wanted: always the two-stage reduction, with the reflectors of stage 1 and a copy of the band kept
    const int bw = lead->nb > 0 ? band_width(lead->nb) : auto_band_width(n2);
    const BatchRef kv = R(L.Vall, mat), kt2 = R(L.Tall, (long long)n2 * 32);
    nl += bsk::launch_sy2sb(n2, n2, bw, R(L.Ak, mat), R(L.VW, L.vw_stride), R(L.SM, L.sm_stride), R(L.AB, L.ab_stride),
                            ncells, nk, s, &kv, &kt2);
    bsk::launch_copy_matrix(2 * bw, n2, R(L.AB, L.ab_stride), 2 * bw, R(L.AB2, L.ab_stride), 2 * bw, ncells, nk, s); ++nl;
    bsk::launch_sb2st(n2, bw, R(L.AB, L.ab_stride), d, e, ncells, nk, s, false, 0, chase_sync); ++nl;
  } else if (lead->algo == BS_TRIDIAG_ONE_STAGE) {
    nl += bsk::launch_tridiag(n2, n2, lead->nb > 0 ? lead->nb : 32, R(L.Ak, mat), R(L.VW, L.vw_stride),
                              R(L.P, (long long)bsk::tridiag_p_elems(n2)), d, e, scal, ncells, nk, s);  // S6
  } else if (n2 <= bsk::tridiag_small_max_n()) {
    bsk::launch_tridiag_small(n2, n2, R(L.Ak, mat), d, e, ncells, nk, s); ++nl;                        // S6, matrix in shared memory
  } else {
    const int bw = lead->nb > 0 ? band_width(lead->nb) : auto_band_width(n2);
    nl += bsk::launch_sy2sb(n2, n2, bw, R(L.Ak, mat), R(L.VW, L.vw_stride), R(L.SM, L.sm_stride), R(L.AB, L.ab_stride),
                            ncells, nk, s);                                                             // S6 stage 1
    bsk::launch_sb2st(n2, bw, R(L.AB, L.ab_stride), d, e, ncells, nk, s, lead->algo == BS_TRIDIAG_TWO_STAGE_STREAMED, 0,
                      chase_sync); ++nl;                         // S6 stage 2
  }
  tick(lead, 2, s);
  bsk::launch_sturm(n2, d, e, nbands, lam, (int)nmat, s, lead->out_root != 0); ++nl;                                       // S7
  tick(lead, 3, s);
  lead->launches += nl;
  lead->last_n = n2; lead->last_nmat = (int)nmat; lead->last_nk = nk;
  lead->last_lam = lam;
  // S8: one copy of ncells x nk x nbands doubles
  cudaPointerAttributes attr;
  bool on_device = false;
  if (cudaPointerGetAttributes(&attr, omega2_out) == cudaSuccess) on_device = attr.type == cudaMemoryTypeDevice;
  else cudaGetLastError();
  CU(cudaMemcpyAsync(omega2_out, lam, nmat * nbands * sizeof(double),
                     on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
  if (!on_device || lead->timing) CU(cudaStreamSynchronize(s));
  if (bsk::g_kt) bsk::g_kt->collect();
  if (lead->timing) {
    lead->ms[BS_T_PENCIL] = tock(lead, 0, 1);
    lead->ms[BS_T_TRIDIAG] = tock(lead, 1, 2);
    lead->ms[BS_T_BISECT] = tock(lead, 2, 3);
  }
  CU(cudaGetLastError());
  return BS_OK;
}

bs_status bs_bands(bs_cell *cell, int32_t nk, const double *kpts, int32_t nbands, double *omega2_out, void *stream) {
  if (!cell) return fail(BS_ERR_ARG, "bs_bands: null handle");
  return bs_bands_batch(&cell, 1, nk, kpts, nbands, omega2_out, stream);
}

// Copies `count` blocks of `block` complex elements with source pitch `src_pitch` (elements) to a dense destination on the
// host or the device.
static bs_status copy_blocks(void *dst, const cplx *src, size_t block, size_t src_pitch, size_t count, cudaStream_t s) {
  cudaPointerAttributes attr;
  bool on_device = false;
  if (cudaPointerGetAttributes(&attr, dst) == cudaSuccess) on_device = attr.type == cudaMemoryTypeDevice;
  else cudaGetLastError();
  CU(cudaMemcpy2DAsync(dst, block * sizeof(cplx), src, src_pitch * sizeof(cplx), block * sizeof(cplx), count,
                       on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
  return BS_OK;
}

bs_status bs_modes_batch(bs_cell *const *cells, int32_t ncells, int32_t nk, const double *kpts, int32_t nbands,
                         double *omega2_out, void *U_out, void *S_out, void *stream) {
  if (!cells || ncells < 1 || !cells[0] || !kpts || !omega2_out || (!U_out && !S_out)) return fail(BS_ERR_ARG, "bs_modes: null argument");
  bs_cell *cell = cells[0];  // the lead: options are equal across the batch (checked by bs_bands_batch)
  if (cell->nvmax < 1) return fail(BS_ERR_STATE, "bs_modes: set BS_OPT_MODES (before sizing the workspace and bs_assemble) first");
  if (nbands < 1 || nbands > cell->nvmax) return fail(BS_ERR_ARG, "bs_modes: nbands must be in 1..BS_OPT_MODES = %d", cell->nvmax);
  if (cell->out_root) return fail(BS_ERR_STATE, "bs_modes: needs BS_OPT_OUTPUT = BS_OUTPUT_OMEGA2");
  cudaStream_t s = (cudaStream_t)stream;
  // S4..S7 with the reflectors of stage 1 and the band kept
  cell->keep_modes = true;
  bs_status st = bs_bands_batch(cells, ncells, nk, kpts, nbands, omega2_out, stream);
  cell->keep_modes = false;
  if (st != BS_OK) return st;
  const int Mt = cell->lay.Mt;
  const Layout L = make_layout(Mt, nk, cell->mode, cell->nb, cell->nvmax);
  const int N = L.N, n2 = 2 * N, n3 = 3 * N, nv = cell->nvmax;
  const int bw = cell->nb > 0 ? band_width(cell->nb) : auto_band_width(n2);
  auto R = [&](long long off, long long stride = 0) { return ref(cell, ncells, cells, off, stride); };
  const long long zs = (long long)n2 * nv;
  int64_t nl = 0;
  // 1. eigenvectors of the band matrix by inverse iteration at the eigenvalues of S7
  bsk::launch_band_invit(n2, bw, R(L.AB2, L.ab_stride), cell->last_lam, nbands, R(L.Zv, zs), R(L.LU, L.lu_stride), ncells, nk, s); ++nl;
  // 2. back through the block reflectors of stage 1, last panel first: Z[r0:] -= V (T (V^H Z[r0:]))
  int c_last = -1;
  for (int c0 = 0; c0 + bw < n2 - 1; c0 += bw) c_last = c0;
  for (int c0 = c_last; c0 >= 0; c0 -= bw) {
    const int r0 = c0 + bw, m = n2 - r0;
    bsk::GemmDesc g{};
    g.ncells = ncells; g.inner = nk; g.kclass = bsk::KC_OTHER;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    g.M = bw; g.N = nbands; g.K = m; g.opA = 1; g.opB = 0;
    g.A = R(L.Vall + (long long)c0 * n2 + r0, (long long)n2 * n2); g.lda = n2;
    g.B = R(L.Zv + r0, zs); g.ldb = n2;
    g.C = R(L.Wa, 32LL * nv); g.ldc = bw;
    bsk::launch_zgemm(g, s);
    g.M = bw; g.N = nbands; g.K = bw; g.opA = 0;
    g.A = R(L.Tall + (long long)(c0 / bw) * bw * bw, (long long)n2 * 32); g.lda = bw;
    g.B = R(L.Wa, 32LL * nv); g.ldb = bw;
    g.C = R(L.Wb, 32LL * nv); g.ldc = bw;
    bsk::launch_zgemm(g, s);
    g.M = m; g.N = nbands; g.K = bw;
    g.A = R(L.Vall + (long long)c0 * n2 + r0, (long long)n2 * n2); g.lda = n2;
    g.B = R(L.Wb, 32LL * nv); g.ldb = bw;
    g.C = R(L.Zv + r0, zs); g.ldc = n2;
    g.alpha = cmake(-1.0, 0.0); g.beta = cmake(1.0, 0.0);
    bsk::launch_zgemm(g, s);
    nl += 3;
  }
  // 3. U = L_Psi^-H y = diag(X_R^H, X_R^H) y   (U^H Psi U = y^H y = I)
  for (int blk = 0; blk < 2; ++blk) {
    bsk::GemmDesc g{};
    g.ncells = ncells; g.inner = nk; g.kclass = bsk::KC_OTHER;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    g.M = N; g.N = nbands; g.K = N; g.opA = 1; g.opB = 0;
    g.A = R(L.XR, 0); g.lda = N;
    g.B = R(L.Zv + (long long)blk * N, zs); g.ldb = n2;
    g.C = R(L.Uv + (long long)blk * N, zs); g.ldc = n2;
    bsk::launch_zgemm(g, s); ++nl;
  }
  // 4. S = Phi^-1 H U with H = V B(k) (the paper's S = -Phi^-1 H* U; its H* is -H, R3)
  if (S_out || cell->refine) {
    std::vector<double> kv((size_t)nk * 2 * N);
    const int W = 2 * Mt + 1;
    for (int c = 0; c < ncells; ++c) {  // (k + G) in Cartesian components, per cell: [k][x | y][N] doubles in its workspace
      for (int k = 0; k < nk; ++k)
        for (int a1 = -Mt; a1 <= Mt; ++a1)
          for (int a2 = -Mt; a2 <= Mt; ++a2) {
            const int g = (a1 + Mt) * W + (a2 + Mt);
            const double f1 = kpts[2 * k] + a1, f2 = kpts[2 * k + 1] + a2;
            kv[((size_t)k * 2 + 0) * N + g] = f1 * cells[c]->Q[0] + f2 * cells[c]->Q[2];
            kv[((size_t)k * 2 + 1) * N + g] = f1 * cells[c]->Q[1] + f2 * cells[c]->Q[3];
          }
      // (pageable source: the copy is staged before the call returns, so kv may be refilled for the next cell)
      CU(cudaMemcpyAsync((cplx *)cells[c]->ws + L.kapm, kv.data(), kv.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    }
    const long long hs = (long long)n3 * nv;
    bsk::launch_apply_h(N, cell->V, R(L.Uv, zs), n2, R(L.HU, hs), n3, R(L.kapm, N), nbands, ncells, nk, s); ++nl;
    bsk::GemmDesc g{};
    g.ncells = ncells; g.inner = nk; g.kclass = bsk::KC_OTHER;
    g.alpha = cmake(1.0, 0.0); g.beta = cmake(0.0, 0.0);
    g.M = n3; g.N = nbands; g.K = n3; g.opA = 0; g.opB = 0;
    g.A = R(L.Y, 0); g.lda = n3;
    g.B = R(L.HU, hs); g.ldb = n3;
    g.C = R(L.Sv, hs); g.ldc = n3;
    bsk::launch_zgemm(g, s); ++nl;
    for (int c = 0; S_out && c < ncells; ++c) {
      st = copy_blocks((cplx *)S_out + (size_t)c * nk * n3 * nbands, (cplx *)cells[c]->ws + L.Sv, (size_t)n3 * nbands, (size_t)hs, nk, s);
      if (st != BS_OK) return st;
    }
    if (cell->refine) {
      // 5. omega^2 again, as the Rayleigh quotient (H u)^dagger Phi^-1 (H u) / (y^dagger y) of every mode (BS_OPT_REFINE)
      bsk::launch_rayleigh(n3, n2, R(L.HU, hs), R(L.Sv, hs), n3, R(L.Zv, zs), n2, cell->last_lam, nbands, ncells, nk, s); ++nl;
      cudaPointerAttributes attr;
      bool on_device = false;
      if (cudaPointerGetAttributes(&attr, omega2_out) == cudaSuccess) on_device = attr.type == cudaMemoryTypeDevice;
      else cudaGetLastError();
      CU(cudaMemcpyAsync(omega2_out, cell->last_lam, (size_t)ncells * nk * nbands * sizeof(double),
                         on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
    }
  }
  for (int c = 0; U_out && c < ncells; ++c) {
    st = copy_blocks((cplx *)U_out + (size_t)c * nk * n2 * nbands, (cplx *)cells[c]->ws + L.Uv, (size_t)n2 * nbands, (size_t)zs, nk, s);
    if (st != BS_OK) return st;
  }
  cell->launches += nl;
  CU(cudaStreamSynchronize(s));
  CU(cudaGetLastError());
  return BS_OK;
}

bs_status bs_modes(bs_cell *cell, int32_t nk, const double *kpts, int32_t nbands, double *omega2_out, void *U_out, void *S_out,
                   void *stream) {
  if (!cell) return fail(BS_ERR_ARG, "bs_modes: null argument");
  return bs_modes_batch(&cell, 1, nk, kpts, nbands, omega2_out, U_out, S_out, stream);
}

bs_status bs_get_tridiagonal(bs_cell *c, double *d_host, double *e_host) {
  if (!c || !d_host || !e_host) return fail(BS_ERR_ARG, "bs_get_tridiagonal: null argument");
  if (!c->d_flat || c->last_nmat == 0) return fail(BS_ERR_STATE, "bs_get_tridiagonal: no bs_bands call led by this handle yet");
  const size_t cnt = (size_t)c->last_nmat * c->last_n;
  sync_handle(c);
  CU(cudaMemcpy(d_host, c->d_flat, cnt * sizeof(double), cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(e_host, c->d_flat + cnt, cnt * sizeof(double), cudaMemcpyDeviceToHost));
  return BS_OK;
}

// ---------------------------------------------------------------- diagnostics: building blocks on caller-owned device arrays
static BatchRef raw(const void *p, long long stride) {
  BatchRef r;
  r.bases = nullptr; r.single = (unsigned long long)p; r.off = 0; r.stride = stride;
  return r;
}

bs_status bs_zgemm(int32_t opA, int32_t opB, int32_t M, int32_t N, int32_t K, const double alpha[2], const void *A,
                   int32_t lda, int64_t strideA, const void *B, int32_t ldb, int64_t strideB, const double beta[2],
                   void *C, int32_t ldc, int64_t strideC, int32_t batch, int32_t flags, void *stream) {
  if (!A || !B || !C || !alpha || !beta || M < 0 || N < 0 || K < 0 || batch < 1) return fail(BS_ERR_ARG, "bs_zgemm: bad argument");
  if ((flags & BS_GEMM_A_HERM_LOWER) && (opA || opB || K != M)) return fail(BS_ERR_ARG, "bs_zgemm: HERM_LOWER needs opA = opB = 0 and K = M");
  bsk::GemmDesc g{};
  g.M = M; g.N = N; g.K = K; g.opA = opA; g.opB = opB; g.lda = lda; g.ldb = ldb; g.ldc = ldc; g.flags = flags;
  g.ncells = 1; g.inner = batch;
  g.alpha = cmake(alpha[0], alpha[1]); g.beta = cmake(beta[0], beta[1]);
  g.A = raw(A, strideA); g.B = raw(B, strideB); g.C = raw(C, strideC);
  bsk::launch_zgemm(g, (cudaStream_t)stream);
  CU(cudaGetLastError());
  return BS_OK;
}

bs_status bs_zpotrf_trtri(int32_t n, void *A, int32_t lda, int64_t strideA, void *X, void *tmp, void *dinv, int32_t *info,
                          int32_t batch, void *stream) {
  if (!A || !X || !tmp || !dinv || !info || n < 1 || batch < 1) return fail(BS_ERR_ARG, "bs_zpotrf_trtri: bad argument");
  cudaStream_t s = (cudaStream_t)stream;
  CU(cudaMemsetAsync(info, 0, sizeof(int) * batch, s));
  // the factor kernels index matrices by cell; express the batch as `batch` cells through a device array of bases
  std::vector<unsigned long long> hb(4 * (size_t)batch);
  const long long dstride = (long long)((n + 63) / 64) * 4096;
  for (int b = 0; b < batch; ++b) {
    hb[b] = (unsigned long long)((cplx *)A + (long long)b * strideA);
    hb[batch + b] = (unsigned long long)((cplx *)X + (long long)b * strideA);
    hb[2 * batch + b] = (unsigned long long)((cplx *)tmp + (long long)b * strideA);
    hb[3 * batch + b] = (unsigned long long)((cplx *)dinv + (long long)b * dstride);
  }
  unsigned long long *db = nullptr;
  CU(cudaMalloc(&db, sizeof(unsigned long long) * hb.size()));
  CU(cudaMemcpyAsync(db, hb.data(), sizeof(unsigned long long) * hb.size(), cudaMemcpyHostToDevice, s));
  auto br = [&](int which) { BatchRef r; r.bases = db + (size_t)which * batch; r.single = 0; r.off = 0; r.stride = 0; return r; };
  bsk::potrf_trtri(n, lda, br(0), br(1), br(2), br(3), info, 0, batch, 1, s);
  CU(cudaStreamSynchronize(s));
  cudaFree(db);
  CU(cudaGetLastError());
  return BS_OK;
}

size_t bs_zhetrd_scratch_elems(int32_t n, int32_t nb) {
  if (n < 1) return 0;
  if (nb < 4) nb = 4;
  if (nb > 32) nb = 32;
  const int bw = band_width(nb);
  return std::max(bsk::tridiag_vw_elems(n, nb), bsk::band_vw_elems(n, bw)) + bsk::tridiag_p_elems(n) +
         align16((long long)bsk::band_sm_elems(bw)) + align16((long long)bsk::band_ab_elems(n, bw)) + 16;
}

bs_status bs_zhetrd(int32_t n, void *A, int32_t lda, int64_t strideA, double *d, double *e, void *scratch, int32_t nb,
                    int32_t algo, int32_t batch, void *stream) {
  if (!A || !d || !e || !scratch || n < 1 || n > 2048 || batch < 1 || lda < n) return fail(BS_ERR_ARG, "bs_zhetrd: bad argument");
  if (nb < 4) nb = 4;
  if (nb > 32) nb = 32;
  // test knob: bits 8.. of algo = the number of sweeps per train of the streamed chase (0: the launcher's choice)
  const int force_g = (algo >> 8) & 0xff;
  algo &= 0xff;
  const int bw = band_width(nb);
  const long long vw = (long long)std::max(bsk::tridiag_vw_elems(n, nb), bsk::band_vw_elems(n, bw));
  const long long pp = (long long)bsk::tridiag_p_elems(n);
  const long long smn = align16((long long)bsk::band_sm_elems(bw)), abn = align16((long long)bsk::band_ab_elems(n, bw));
  const long long per = (long long)bs_zhetrd_scratch_elems(n, nb);
  cplx *sc = (cplx *)scratch;
  BatchRef VW = raw(sc, per), P = raw(sc + vw, per);
  if (algo == BS_TRIDIAG_TWO_STAGE && n <= bsk::tridiag_small_max_n()) {
    bsk::launch_tridiag_small(n, lda, raw(A, strideA), d, e, 1, batch, (cudaStream_t)stream);
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    CU(cudaGetLastError());
    return BS_OK;
  }
  if (algo == BS_TRIDIAG_TWO_STAGE || algo == BS_TRIDIAG_TWO_STAGE_STREAMED) {
    BatchRef SMr = raw(sc + vw + pp, per), ABr = raw(sc + vw + pp + smn, per);
    int *sync = nullptr;
    CU(cudaMalloc(&sync, sizeof(int) * bsk::sb2st_sync_ints(n, batch)));
    bsk::launch_sy2sb(n, lda, bw, raw(A, strideA), VW, SMr, ABr, 1, batch, (cudaStream_t)stream);
    bsk::launch_sb2st(n, bw, ABr, d, e, 1, batch, (cudaStream_t)stream, algo == BS_TRIDIAG_TWO_STAGE_STREAMED, force_g, sync);
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    cudaFree(sync);
    CU(cudaGetLastError());
    return BS_OK;
  }
  // tau of the pending reflector: the 16 spare elements of matrix 0's slot hold nothing else; use a strided view
  // (scal is indexed [2*z]), so place it after all per-matrix slots is not possible without more memory: use slot tails.
  double *scal = nullptr;
  CU(cudaMalloc(&scal, sizeof(double) * 2 * batch));
  bsk::launch_tridiag(n, lda, nb, raw(A, strideA), VW, P, d, e, scal, 1, batch, (cudaStream_t)stream);
  CU(cudaStreamSynchronize((cudaStream_t)stream));
  cudaFree(scal);
  CU(cudaGetLastError());
  return BS_OK;
}

// ---- bs_zhetrd_static: the two-stage tridiagonalisation with its scratch in a static device array ----------------
// For callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).  The array is
// part of the library image: every GPU that loads libbs.so holds BS_ZHETRD_STATIC_BYTES of it until the process exits.
// In host code the NAME of the array is a host-side stand-in, not a device address; the address on the current device
// comes from cudaGetSymbolAddress (once per device, with that device current) and only that pointer goes to kernels.
static __device__ __align__(256) unsigned char g_zhetrd_static[BS_ZHETRD_STATIC_BYTES];

static bs_status zhetrd_static_base(unsigned char **base) {
  static unsigned char *cache[64] = {nullptr};
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(BS_ERR_ARG, "bs_zhetrd_static: device index beyond 63");
  if (!cache[dev]) {
    unsigned char *ptr = nullptr;
    CU(cudaGetSymbolAddress((void **)&ptr, g_zhetrd_static));  // address on the CURRENT device
    if (!ptr) return fail(BS_ERR_CUDA, "bs_zhetrd_static: cudaGetSymbolAddress returned a null pointer");
    cache[dev] = ptr;
  }
  *base = cache[dev];
  return BS_OK;
}

size_t bs_zhetrd_static_bytes(int32_t n, int32_t batch) {
  if (n < 1 || batch < 1) return 0;
  const size_t per = bs_zhetrd_scratch_elems(n, 16) * sizeof(cplx);
  const size_t sync = (sizeof(int) * bsk::sb2st_sync_ints(n, batch) + 255) / 256 * 256;
  return per * (size_t)batch + sync;
}

bs_status bs_zhetrd_static(int32_t n, void *A, int32_t lda, int64_t strideA, double *d, double *e, int32_t batch,
                           void *stream) {
  if (!A || !d || !e || n < 1 || n > 2048 || batch < 1 || lda < n) return fail(BS_ERR_ARG, "bs_zhetrd_static: bad argument");
  const size_t need = bs_zhetrd_static_bytes(n, batch);
  if (need > (size_t)BS_ZHETRD_STATIC_BYTES)
    return fail(BS_ERR_ARG, "bs_zhetrd_static: n = %d, batch = %d needs %zu bytes of scratch, the static array holds %d",
                (int)n, (int)batch, need, (int)BS_ZHETRD_STATIC_BYTES);
  cudaStream_t s = (cudaStream_t)stream;
  if (n <= bsk::tridiag_small_max_n()) {  // the matrix fits in shared memory: no scratch at all
    bsk::launch_tridiag_small(n, lda, raw(A, strideA), d, e, 1, batch, s);
    CU(cudaGetLastError());
    return BS_OK;
  }
  unsigned char *base = nullptr;
  const bs_status st = zhetrd_static_base(&base);
  if (st != BS_OK) return st;
  // layout: [progress words of the chase, padded to 256 B][per-matrix slots as in bs_zhetrd, band width 16]
  const int bw = 16;
  const size_t sync_bytes = (sizeof(int) * bsk::sb2st_sync_ints(n, batch) + 255) / 256 * 256;
  int *sync = reinterpret_cast<int *>(base);
  cplx *sc = reinterpret_cast<cplx *>(base + sync_bytes);
  const long long vw = (long long)std::max(bsk::tridiag_vw_elems(n, bw), bsk::band_vw_elems(n, bw));
  const long long pp = (long long)bsk::tridiag_p_elems(n);
  const long long smn = align16((long long)bsk::band_sm_elems(bw));
  const long long per = (long long)bs_zhetrd_scratch_elems(n, bw);
  BatchRef VW = raw(sc, per), SMr = raw(sc + vw + pp, per), ABr = raw(sc + vw + pp + smn, per);
  // what must start at zero: the progress words (launch_sb2st clears them on the stream) and nothing else: stage 1
  // writes every element of VW / SM / AB that a later kernel of this call reads
  bsk::launch_sy2sb(n, lda, bw, raw(A, strideA), VW, SMr, ABr, 1, batch, s);
  bsk::launch_sb2st(n, bw, ABr, d, e, 1, batch, s, false, 0, sync);
  CU(cudaGetLastError());
  return BS_OK;
}

bs_status bs_sturm(int32_t n, const double *d, const double *e, int32_t nev, double *lam, int32_t batch, void *stream) {
  if (!d || !e || !lam || n < 1 || nev < 1 || nev > n || batch < 1) return fail(BS_ERR_ARG, "bs_sturm: bad argument");
  bsk::launch_sturm(n, d, e, nev, lam, batch, (cudaStream_t)stream);
  CU(cudaGetLastError());
  return BS_OK;
}

}  // extern "C"
