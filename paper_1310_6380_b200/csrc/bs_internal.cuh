// Internal declarations shared by the translation units of libbs.so (sm_100a).  Not part of the C-ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>

#include "bs.h"

typedef double2 cplx;

// ---------------------------------------------------------------- small complex helpers (device)
__host__ __device__ __forceinline__ cplx cmake(double r, double i) { return make_double2(r, i); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {  // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
// acc += a*b
__device__ __forceinline__ void cfma(cplx &acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
__device__ __forceinline__ void cfmac(cplx &acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(-a.y, b.x, acc.y);
}
// acc -= a*b
__device__ __forceinline__ void cfms(cplx &acc, cplx a, cplx b) {
  acc.x = fma(-a.x, b.x, acc.x);
  acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(-a.x, b.y, acc.y);
  acc.y = fma(-a.y, b.x, acc.y);
}

// ---------------------------------------------------------------- batched pointer addressing
// A "batch" is ncells handles (each with its own workspace base) times `inner` equally strided matrices inside each
// workspace.  blockIdx.z = cell * inner + i  ->  bases[cell] + off + i * stride   (units: complex elements).
struct BatchRef {
  const unsigned long long *bases;  // device array [ncells] of workspace base addresses; nullptr -> `single`
  unsigned long long single;        // used when bases == nullptr
  long long off;                    // element offset inside the workspace
  long long stride;                 // element stride between inner matrices
};
__device__ __forceinline__ cplx *batch_ptr(const BatchRef &r, int cell, int i) {
  unsigned long long b = r.bases ? r.bases[cell] : r.single;
  return reinterpret_cast<cplx *>(b) + r.off + (long long)i * r.stride;
}

// ---------------------------------------------------------------- kernels' host launchers (one per .cu)
namespace bsk {

// cudaFuncAttributeMaxDynamicSharedMemorySize is a PER-DEVICE attribute: set it once per (kernel, device).  `mask` is
// the caller's function-local static (one per kernel instantiation), bit d = done on device d.  A race between two host
// threads only sets the attribute twice.
template <class F>
inline void ensure_dyn_smem(F *kernel, int bytes, unsigned long long &mask) {
  int dev = 0;
  cudaGetDevice(&dev);
  const unsigned long long bit = 1ull << (dev & 63);
  if (!(mask & bit)) {
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    mask |= bit;
  }
}

// Per-kernel-class device timing (BS_OPT_TIMING = 2): CUDA events recorded on the launching stream around every launch
// of a class, summed after the call's final synchronise.  `work` is the ALGORITHMIC work of the class (flops for the
// DMMA classes, bytes for the HBM classes), accumulated on the host at launch time.
enum KClass {
  KC_TABLE = 0, KC_EXPAND, KC_GEMM_FACTOR, KC_GEMM_REDUCE, KC_GEMM_TRIDIAG, KC_HEMV, KC_PANEL, KC_STURM, KC_PENCIL,
  KC_COMBINE, KC_POTRF_DIAG, KC_OTHER, KC_BULGE, KC_GEMM_HEMM, KC_GEMM_WY, KC_TRIDIAG_SMALL, KC_COUNT
};
struct KTimer {
  std::vector<cudaEvent_t> ev;   // pool; pairs (2i, 2i+1)
  std::vector<int> cls;          // class of pair i
  size_t used = 0;               // events used
  double work[KC_COUNT] = {0};
  double ms[KC_COUNT] = {0};
  long long count[KC_COUNT] = {0};
  void begin(int c, cudaStream_t s) {
    if (used + 2 > ev.size()) {
      const size_t old = ev.size();
      ev.resize(old + 1024);
      for (size_t i = old; i < ev.size(); ++i) cudaEventCreate(&ev[i]);
    }
    cls.resize(used / 2 + 1);
    cls[used / 2] = c;
    cudaEventRecord(ev[used], s);
  }
  void end(cudaStream_t s) { cudaEventRecord(ev[used + 1], s); used += 2; }
  void reset() {
    used = 0;
    for (int i = 0; i < KC_COUNT; ++i) { work[i] = 0; ms[i] = 0; count[i] = 0; }
  }
  void collect() {  // call after the stream has been synchronised
    for (size_t i = 0; i + 1 < used; i += 2) {
      float t = 0.f;
      cudaEventElapsedTime(&t, ev[i], ev[i + 1]);
      ms[cls[i / 2]] += t;
      count[cls[i / 2]] += 1;
    }
    used = 0;
  }
  ~KTimer() { for (auto e : ev) cudaEventDestroy(e); }
};
extern thread_local KTimer *g_kt;  // nullptr unless the current call runs with BS_OPT_TIMING = 2
struct KScope {                    // RAII: times one launch of class c on stream s and credits `work` to it
  cudaStream_t s; bool on;
  KScope(int c, double work, cudaStream_t st) : s(st), on(g_kt != nullptr) {
    if (on) { g_kt->work[c] += work; g_kt->begin(c, s); }
  }
  ~KScope() { if (on) g_kt->end(s); }
};

struct Geometry {  // device pointers, per cell
  const double *edge;   // SoA [6][nes]: mh1, mh2 (fractional midpoint), eh1, eh2 (fractional edge), ex, ey (Cartesian edge);
                        // nes = nedge rounded up to even: every array starts 16-byte aligned (1-D bulk TMA copies)
  const int *ephase;    // [nedge] phase of each edge
  const double *w;      // [7][P] channel weights: Dv11 Dv22 Dv12 Dv13 Dv23 Dv33 rho
  const double *area;   // [3][P]: signed area, fractional centroid (ch1, ch2)
  int nedge, nes, P;
  double Q[4];          // rows q^1, q^2 (Cartesian)
};

// S1: table[c][(D1+2Mt)*(4Mt+1) + (D2+2Mt)], c < 7.  geo: device array [ncells]; table at BatchRef (inner unused).
// maxP: the largest phase count of the batch (shared memory of the TMA-staged kernel)
// scratch: per cell, scratch_elems complex elements that nothing else uses during S1 (the separable-phase table of
// 4 (4Mt+1) max_nes elements goes there when it fits; otherwise the direct kernels run)
int launch_table(const Geometry *geo_dev, int ncells, int Mt, BatchRef table, double total_edges, int centroid_rule,
                  cudaStream_t s, int maxP, int max_nes, BatchRef scratch, long long scratch_elems);
// S1 for cells that share one geometry: Iph[p + dh * P] = I_p(q_D) once per geometry (poff: device [P+1] edge offsets of
// the phases), then every cell's table as W (7 ncells x P) times Iph on the DMMA GEMM.  W, Tst: device scratch of
// 7 ncells x P and 7 ncells x nhalf complex, nhalf = ((4Mt+1)^2 + 1) / 2.
void launch_phase_table(const Geometry &g, const int *poff, int Mt, cplx *Iph, int centroid_rule, cudaStream_t s);
void launch_shared_tables(const Geometry *geos_dev, int ncells, int P, int Mt, const cplx *Iph, cplx *W, cplx *Tst,
                          BatchRef table, cudaStream_t s);
// S2: Phi (3N x 3N full) and R (N x N full) from the table.
void launch_expand(int ncells, int Mt, BatchRef table, BatchRef Phi, BatchRef R, cudaStream_t s);

// Isotropic shortcut of S3: E = A + B, F = A - B (N x N) from the table; Y from Ei = E^{-1}, Fi = F^{-1}.
void launch_expand_sumdiff(int ncells, int Mt, BatchRef table, BatchRef E, BatchRef F, cudaStream_t s);
void launch_compose_y(int ncells, int N, BatchRef Ei, BatchRef Fi, BatchRef Y, cudaStream_t s);

struct GemmDesc {
  int M, N, K, opA, opB, lda, ldb, ldc, flags, inner, ncells;
  int kclass;  // KClass the launch is timed under (0 -> KC_OTHER)
  int ksplit;  // > 1: split K into ksplit chunks, chunk s writes its partial product to C + s * split_stride (beta ignored)
  long long split_stride;
  cplx alpha, beta;
  BatchRef A, B, C;
};
void launch_zgemm(const GemmDesc &g, cudaStream_t s);

// S3 pieces.  A: n x n (lda) lower Cholesky in place; X = L^{-1}; tmp same shape as A; dinv: ceil(n/64) blocks of 64x64.
// info: device int per (cell*inner).  Returns number of kernel launches issued.
int potrf_trtri(int n, int lda, BatchRef A, BatchRef X, BatchRef tmp, BatchRef dinv, int *info, long long info_stride_unused,
                int ncells, int inner, cudaStream_t s);
void launch_copy_matrix(int rows, int cols, BatchRef src, int lds, BatchRef dst, int ldd, int ncells, int inner,
                        cudaStream_t s);
void launch_hermitian_fill_upper(int n, BatchRef A, int lda, int ncells, int inner, cudaStream_t s);

// S4: K = V^2 sum_t Btilde(kL_t)^T Y Btilde(kR_t), nterm <= 2.  kvec: per output matrix
// (cell, i) doubles [nterm][2 (L,R)][2 (x,y)][N] at the BatchRef (offset/stride in complex elements = 2 doubles).
void launch_pencil(int N, double V2, BatchRef Y, int ldy, BatchRef K, int ldk, BatchRef kvec, int nterm, int ncells,
                   int inner, cudaStream_t s);
// A(k) = sum_i c_i(k) Coef_i, lower triangle (by 64-tiles) only.  coef: [ncells*nk][6] doubles.
void launch_combine(int n, BatchRef Coef, long long coef_mat_stride, BatchRef Ak, int ld, const double *coefk, int nk,
                    int ncells, cudaStream_t s);

// S6: tridiagonalisation (lower triangle of A read; A22 blocks overwritten).  VW: per matrix tridiag_vw_elems complex,
// P: per matrix tridiag_p_elems complex (hemv partial sums), d,e: per matrix n doubles at d + z*n, scal: 2 doubles per
// matrix.  Returns the number of kernel launches issued.
size_t tridiag_vw_elems(int n, int nb);
size_t tridiag_p_elems(int n);
int launch_tridiag(int n, int lda, int nb, BatchRef A, BatchRef VW, BatchRef P, double *d, double *e, double *scal,
                   int ncells, int inner, cudaStream_t s);
// S6, two-stage (band.cu, bulge.cu): dense -> band of width b (b in {8,16,32}) -> tridiagonal.
// VW: per matrix band_vw_elems, SM: per matrix band_sm_elems, AB: per matrix band_ab_elems complex.
size_t band_vw_elems(int n, int b);
size_t band_sm_elems(int b);
size_t band_ab_elems(int n, int b);
// keepV / keepT (optional, for the mode shapes): the reflectors of every panel are also stored, V of the panel at columns
// c0 .. c0+b-1 in keepV (n x n per matrix, ld n, rows r0 .. n-1 written) and its compact-WY T in keepT + (c0 / b) b^2.
int launch_sy2sb(int n, int lda, int b, BatchRef A, BatchRef VW, BatchRef SM, BatchRef AB, int ncells, int inner,
                 cudaStream_t s, const BatchRef *keepV = nullptr, const BatchRef *keepT = nullptr);
// streamed: stream the band through the ring even when it would fit shared memory; force_g > 0: at most that many
// sweeps per train (test knob); sync: device scratch of sb2st_sync_ints(n, nmat) ints (task counter + train progress)
void launch_sb2st(int n, int b, BatchRef AB, double *d, double *e, int ncells, int inner, cudaStream_t s, bool streamed,
                  int force_g, int *sync);
size_t sb2st_sync_ints(int n, int nmat);
bool bulge_band_resident(int n, int b);  // stage 2 keeps the whole band of width b in shared memory
// S6 for n <= tridiag_small_max_n(): the matrix in shared memory, one CTA per matrix, unblocked Householder (small.cu).
int tridiag_small_max_n();
void launch_tridiag_small(int n, int lda, BatchRef A, double *d, double *e, int ncells, int inner, cudaStream_t s);
// Mode shapes (modes.cu): inverse iteration on the Hermitian band matrix (width b, ld 2b) for the nvec eigenvalues lam
// (nvec per matrix, ascending), Z: n x nvec per matrix (ld n), LU: band_invit_lu_elems(n, b) complex of scratch per matrix.
size_t band_invit_lu_elems(int n, int b);
void launch_band_invit(int n, int b, BatchRef AB, const double *lam, int nvec, BatchRef Z, BatchRef LU, int ncells, int inner,
                       cudaStream_t s);
// HU = V B(k) U (3N x nvec from 2N x nvec); kap: per matrix [2][N] doubles (kx, ky of k + G).
void launch_apply_h(int N, double V, BatchRef U, int ldu, BatchRef HU, int ldh, BatchRef KAP, int nvec, int ncells,
                    int inner, cudaStream_t s);  // KAP: per matrix [kx | ky][N] doubles (stride N complex elements)
// out[z * nvec + j] = Re (HU_j^dagger S_j) / (Y_j^dagger Y_j): the factored Rayleigh quotient of mode j of matrix z
void launch_rayleigh(int n3, int n2, BatchRef HU, BatchRef S, int lds, BatchRef Y, int ldy, double *out, int nvec, int ncells,
                     int inner, cudaStream_t s);
// S7: Sturm bisection.  lam: per matrix nev doubles at lam + z*nev.
void launch_sturm(int n, const double *d, const double *e, int nev, double *lam, int nmat, cudaStream_t s,
                  bool root = false);  // root: write sqrt(max(lambda, 0)) instead of lambda

}  // namespace bsk
