// rt_api.cu -- the C ABI of include/rt_tddft.h: context, workspaces, the step schedule, getters.
// Everything numerical happens in the kernels of gemm_kernels.cu / grid_kernels.cu; this file only owns
// memory, enqueues launches in the order of Algorithm 1 and moves results across the ABI.
#include "../../include/rt_tddft.h"
#include "rt_internal.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <queue>
#include <string>
#include <vector>

using namespace rt;

namespace {

thread_local std::string g_create_error = "";

struct EventPair { cudaEvent_t a, b; int stage; };

}  // namespace

struct rt_ctx {
  rt_config cfg{};
  int N = 0, ldn = 0;
  long long Ng = 0;              // points of the whole grid
  long long Ngl = 0;             // points this handle's Phi covers (= Ng unless the handle is a grid slab)
  long long slab_off = 0;        // first grid point of the slab
  int x0 = 0;                    // first x-plane of the slab
  bool slab = false;
  int slab_state = 0;            // 0: waiting for RT_SLAB_INIT, 1: ready
  int hist_cap = 0;              // dipole history (time levels kept on the device); 0 = off
  double* d_hist = nullptr;      // [hist_cap][4]
  unsigned long long* d_hist_n = nullptr;   // levels recorded so far (device counter: the step graph increments it)
  int64_t steps_done = 0;        // time levels after t = 0 enqueued so far
  int64_t hist_first = 0;        // oldest level the history can hold (0, or the level restored by rt_set_state)
  double theta0 = 0;             // dt * (spectral half-width + 0.5 Ha margin): the series orders were sized with this
  double half_len[3] = {0, 0, 0}; // largest |x_q| on the grid
  double* op_T[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // rt_op_propagate scratch (lazily allocated once)
  GridDims gd{};
  double h = 0, dvol = 0, dt = 0, sigma = 0, omega = 0;
  int m = 2, n_vc = 0, nu1 = 2, nu2 = 2, q = 0;           // q: cos/sinc polynomial degree in Y = X^2
  bool use_h = true, use_xc = true, use_graph = true;
  cudaStream_t st = nullptr;
  bool poisoned = false;
  std::string err;
  double t = 0;
  int64_t launches = 0;          // kernels enqueued so far
  int64_t launches_per_step = 0;

  const double* phi = nullptr;   // borrowed or owned
  double* phi_owned = nullptr;
  std::vector<void*> allocs;

  // N-vectors / scalars
  double *d_eps = nullptr, *d_occ = nullptr, *d_E = nullptr, *d_sums = nullptr, *d_bsums = nullptr, *d_energy = nullptr;
  // N x N (ld = ldn)
  double *Hm1 = nullptr, *H0 = nullptr, *H1 = nullptr, *X = nullptr, *Ya = nullptr, *Yb = nullptr, *Yc = nullptr,
         *Cm = nullptr, *Sc = nullptr, *Sm = nullptr, *P0r = nullptr, *P0i = nullptr, *P1r = nullptr, *P1i = nullptr,
         *W = nullptr;
  int2* d_tiles = nullptr;        // upper tiles (ti <= tj), class-ordered and 2-D blocked for the projection
  int2* d_tiles_full = nullptr;   // all ntile x ntile tiles, row-major (a row block of the sharded propagator is a contiguous piece)
  int2* d_tiles_sym = nullptr;    // upper tiles (ti <= tj) row-major: the symmetric-output N x N GEMMs (stream-K walks them in order)
  int ntile = 0;
  double* gemm_ws = nullptr;      // stream-K fix-up workspace and flags of the TMA N x N GEMM (gemm_tma.cu)
  std::vector<double*> pw_extra;  // Y^4 .. Y^q of the Taylor propagator (Y^2, Y^3 live in Yb, Yc)
  int* pace_cnt = nullptr;        // checkpoint counters of the paced projection launch (gemm_tma.cu), nullptr: not paced
  int pace_w = 1;                 // how many checkpoints a CTA may lead the slowest one by
  bool dens_resident = false;     // density raster regime (a): fold resident in L2, Phi panels kept with evict_last
  int* gemm_sync = nullptr;
  // row-sharded propagator: rank `shard` of `nshard` owns the rows [row_beg, row_end) of every N x N product
  int nshard = 1, shard = 0, shard_rows = 0, row_beg = 0, row_end = 0;
  size_t nn_alloc = 0;            // doubles per N x N buffer (rows padded to nshard * shard_rows for the all-gathers)
  // closer-to-paper propagation: general Omega = -i dt S^-1 Hbar (+ dt^2/12 [S^-1 H0, S^-1 H1])
  int magnus = 1;                 // 2: second Magnus term (Eq. 13)
  bool nonorth = false;           // RT_NONORTHOGONAL: S = dVol Phi Phi^T != 1 (Eq. 33-38)
  bool general = false;           // magnus == 2 || nonorth: the series runs in the "one multiply + transpose" form
  double *Hks = nullptr;          // ground-state Hamiltonian matrix when it is not diag(eps)   (rt_create_general)
  double *Smat = nullptr, *Sinv = nullptr, *Bm = nullptr, *Wm = nullptr, *Rt = nullptr, *It = nullptr;
  int newton_iters = 0;           // Newton-Schulz iterations that S^-1 took at create
  int xc_kind = RT_XC_LDA_PZ81;   // RT_XC_PBE: GGA with finite-difference gradients (grid_kernels.cu)
  int fd_order = 2;               // order of the grid operators: gradient of the GGA, Laplacian of the Hartree solve
  double *pbe_scr = nullptr, *vxc_cur = nullptr, *exc_a = nullptr, *exc_b = nullptr;     // [4 Ng], [Ng], [Ng], [Ng]
  double *f4 = nullptr;           // right-hand side of the fourth-order Hartree solve
  MgLevel dl0{};                  // level-0 arrays of its correction hierarchy
  int slab_more = 0;              // decision of the last RT_SLAB_CHECK: another Hamiltonian update is needed
  std::map<int, cudaGraphExec_t> phase_exec;      // slab phases captured as CUDA graphs, key = (phase, it == 0, last update)
  std::map<int, int64_t> phase_launches;
  std::map<int, int> phase_capture_failures;      // captures of a phase that were invalidated (the phase then ran directly)
  int capture_failures = 0;
  std::vector<cudaGraph_t> phase_graphs;
  DensSeg* d_segs = nullptr;
  std::vector<DensSeg> segs;
  ProjectPlan pp{};
  DensityPlan dp{};
  // grid arrays
  double *rho = nullptr, *rho0 = nullptr, *vxc0 = nullptr, *w = nullptr, *rho_part = nullptr, *op_u = nullptr;
  std::vector<MgLevel> lv;
  double *Qx = nullptr, *Qy = nullptr, *Qz = nullptr, *lx = nullptr, *ly = nullptr, *lz = nullptr;

  cudaGraph_t graph = nullptr;
  cudaGraphExec_t gexec = nullptr;
  // dynamic-H_thrs mode: one graph per kind of Hamiltonian update (first of a step / later ones)
  cudaGraph_t graph_upd[2] = {nullptr, nullptr};
  cudaGraphExec_t gexec_upd[2] = {nullptr, nullptr};
  int64_t launches_per_upd[2] = {0, 0};

  // the paper's loops (Alg. 1 lines 12-26): commutator series with dP_thrs, Hamiltonian loop with H_thrs
  int prop = RT_PROP_TAYLOR;
  int kmax = 0;
  double dP_thrs = 0, H_thrs = 0;
  int max_hup = 0;
  bool dynamic = false;
  ConvState* d_cs = nullptr;
  int last_hupdates = 0, last_orders = 0;
  double last_H_err = 0, last_dP_err = 0;

  // TMA descriptors: Phi as a K-contiguous operand (box 16 x 128) and as an N-contiguous one (box 16 x 16);
  // one K-contiguous descriptor per library-owned N x N buffer
  bool use_tma = false;
  int sms = 148;
  CUtensorMap tmPhiK{}, tmPhiN{};
  int phiN_3d = 0;
  std::map<const double*, CUtensorMap> tmN;

  bool timing = false;
  std::vector<EventPair> ev_used;
  std::vector<EventPair> ev_free;
  double stage_ms[RT_STAGE_COUNT] = {0, 0, 0, 0, 0};
  int64_t stage_calls[RT_STAGE_COUNT] = {0, 0, 0, 0, 0};
};

namespace {

int fail(rt_ctx* c, int code, const std::string& msg) {
  if (c) { c->err = msg; if (code == RT_ECUDA) c->poisoned = true; }
  else g_create_error = msg;
  return code;
}

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(c, RT_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));                 \
  } while (0)

#define CHECK_HANDLE(c)                                                                            \
  do {                                                                                             \
    if (!(c)) return fail(nullptr, RT_ESTATE, "NULL handle");                                       \
    if ((c)->poisoned) return RT_ESTATE;                                                           \
  } while (0)

template <class T>
int dev_alloc(rt_ctx* c, T** p, size_t count) {
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, count * sizeof(T) > 0 ? count * sizeof(T) : 16);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(c, RT_ENOMEM, std::string("cudaMalloc failed: ") + cudaGetErrorString(e));
  }
  c->allocs.push_back(q);
  *p = reinterpret_cast<T*>(q);
  return RT_OK;
}

int roundup(int x, int m) { return (x + m - 1) / m * m; }
constexpr int BK_HOST = 16;      // doubles per pipeline stage (dmma_core.cuh BK)

// real orthonormal eigenvectors of the periodic 1-D second-difference operator: column 0 constant,
// then (cos_k, sin_k) pairs, then the alternating vector when n is even.  lam[col] = (2 - 2 cos(2 pi k/n))/h^2.
void eigenbasis_1d(int n, double h, std::vector<double>& Q, std::vector<double>& lam) {
  const double PI = 3.14159265358979323846;
  Q.assign((size_t)n * n, 0.0);
  lam.assign(n, 0.0);
  int col = 0;
  for (int i = 0; i < n; ++i) Q[(size_t)i * n + col] = 1.0 / std::sqrt((double)n);
  lam[col++] = 0.0;
  for (int k = 1; 2 * k < n; ++k) {
    const double l = (2.0 - 2.0 * std::cos(2.0 * PI * k / n)) / (h * h);
    for (int i = 0; i < n; ++i) {
      // reduce the angle argument exactly in integers before calling cos/sin
      const long long kk = ((long long)k * i) % n;
      Q[(size_t)i * n + col] = std::sqrt(2.0 / n) * std::cos(2.0 * PI * (double)kk / n);
      Q[(size_t)i * n + col + 1] = std::sqrt(2.0 / n) * std::sin(2.0 * PI * (double)kk / n);
    }
    lam[col] = lam[col + 1] = l;
    col += 2;
  }
  if (n % 2 == 0 && n > 1) {
    for (int i = 0; i < n; ++i) Q[(size_t)i * n + col] = ((i & 1) ? -1.0 : 1.0) / std::sqrt((double)n);
    lam[col++] = 4.0 / (h * h);
  }
}

bool can_coarsen(const GridDims& g) {
  return g.nx % 2 == 0 && g.ny % 2 == 0 && g.nz % 2 == 0 && g.nx > 4 && g.ny > 4 && g.nz > 4;
}

// ---- a5 work types ---------------------------------------------------------------------------------
// The triangular fold leaves j-tile jt with the contraction rows k >= jt*TILE, i.e. nk(jt) stages of 16.  Pair
// (p, ntile-1-p) therefore always costs about (ntile + 1) tiles.  The time line of a pair is: LONG tile p with k
// DESCENDING from N, then short tile ntile-1-p with k ASCENDING to N.  With that order the contraction row a CTA reads
// at stage t of its item does not depend on the pair (first N - 16 (t + 1), then 16 t - (N - 128 (ntile - 1)) ... ): CTAs
// that start their items together read the SAME Phi rows at the same time whatever their type, so the Phi tile of an
// r-tile is fetched from DRAM once for all the types that run beside each other.  (Round 1 / first round-2 order --
// short tile up, then long tile down -- made every type read its own rows: 7.2 TB of DRAM reads per launch at
// N = 13,000, no reuse of Phi between types at all.)  The time line is cut into `nsplit` pieces of equal length; each
// piece is a work type (<= 2 segments) with its own partial-sum row.
// aligned = false keeps the round-1 order (short tile up, then long tile down: the rows around the turn-around are re-read
// while still in L2), which measured better when the Phi panels in flight are held in L2 anyway (regime (a) of the raster
// below: nano 72 GB / 344.9 ms per launch against 280 GB / 351.9 ms with the aligned order).
void build_density_types(int N, int ntile, int nsplit, bool aligned, std::vector<DensSeg>& out) {
  out.clear();
  const int npairs = (ntile + 1) / 2;
  auto nk = [&](int jt) { return (N - jt * TILE + BK_HOST - 1) / BK_HOST; };
  for (int p = 0; p < npairs; ++p) {
    const int jb = ntile - 1 - p;
    const int nkA = nk(p), nkB = jb > p ? nk(jb) : 0;
    const int tot = nkA + nkB;
    for (int i = 0; i < nsplit; ++i) {
      const int t0 = (int)((long long)tot * i / nsplit), t1 = (int)((long long)tot * (i + 1) / nsplit);
      DensSeg a{p, 0, 0, -1}, b{jb > p ? jb : p, 0, 0, 1};
      if (aligned) {                       // long tile down, then short tile up
        if (t0 < nkA) { a.s0 = nkA - 1 - t0; a.ns = (t1 < nkA ? t1 : nkA) - t0; }
        if (t1 > nkA) {
          const int u0 = (t0 > nkA ? t0 : nkA) - nkA, u1 = t1 - nkA;
          b.s0 = u0; b.ns = u1 - u0;
        }
        out.push_back(a);
        out.push_back(b);
      } else {                             // short tile up, then long tile down
        if (t0 < nkB) { b.s0 = t0; b.ns = (t1 < nkB ? t1 : nkB) - t0; }
        if (t1 > nkB) {
          const int u0 = (t0 > nkB ? t0 : nkB) - nkB, u1 = t1 - nkB;
          a.s0 = nkA - 1 - u0; a.ns = u1 - u0;
        }
        out.push_back(b);
        out.push_back(a);
      }
    }
  }
}

// ---- TMA descriptors -------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
    else
      cudaGetLastError();
  }
  return fn;
}
// row-major FP64 matrix [rows][cols] with leading dimension ld (doubles); box = {box_cols, box_rows}; 128B swizzle
bool make_map(CUtensorMap* m, const double* base, long long rows, long long cols, long long ld, int box_cols,
              int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 8};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  cuuint32_t es[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// Phi [N][Ng] viewed as {16 (r low), N (k), Ng/16 (r high)}: one box {16, 16, 8} lands in shared memory as 8
// consecutive [16 k][16 r] sub-tiles, the layout the density kernel's B fragments read
bool make_map_phi3d(CUtensorMap* m, const double* base, long long N, long long Ng) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn || Ng % 16) return false;
  cuuint64_t dims[3] = {16, (cuuint64_t)N, (cuuint64_t)(Ng / 16)};
  cuuint64_t strides[2] = {(cuuint64_t)Ng * 8, 128};
  cuuint32_t box[3] = {16, 16, 8};
  cuuint32_t es[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
const CUtensorMap& nn_map(rt_ctx* c, const double* p) {
  auto it = c->tmN.find(p);
  if (it == c->tmN.end()) {
    CUtensorMap m{};
    make_map(&m, p, c->N, c->N, c->ldn, BK_HOST, TILE);
    it = c->tmN.emplace(p, m).first;
  }
  return it->second;
}

// ---- stage timing helpers ------------------------------------------------------------------------
void stage_begin(rt_ctx* c, int stage) {
  if (!c->timing) return;
  EventPair ep;
  if (!c->ev_free.empty()) { ep = c->ev_free.back(); c->ev_free.pop_back(); }
  else { cudaEventCreate(&ep.a); cudaEventCreate(&ep.b); }
  ep.stage = stage;
  cudaEventRecord(ep.a, c->st);
  c->ev_used.push_back(ep);
}
void stage_end(rt_ctx* c) {
  if (!c->timing) return;
  cudaEventRecord(c->ev_used.back().b, c->st);
}

// ---- the stages ------------------------------------------------------------------------------------
// sym = +1 / -1: D is known to be (anti)symmetric: upper tiles + mirror image.  rows = true: this launch computes only
// the row block [row_beg, row_end) that this rank owns (row-sharded propagator; nshard = 1: the whole matrix) -- as a
// plain product, because the mirror image of a row block belongs to other ranks.
void enqueue_gemm(rt_ctx* c, int sym, const double* A0, const double* B0, double a0, const double* A1,
                  const double* B1, double a1, double* D, double* Z1 = nullptr, double b1 = 0, double* Z2 = nullptr,
                  double b2 = 0, const int* skip = nullptr, bool rows = false) {
  const bool shard = rows && c->nshard > 1;
  GemmArgs g{c->N, c->ldn, A0, B0, a0, A1, B1, a1, D, Z1, b1, Z2, b2, skip, shard ? c->row_beg : 0,
             shard ? c->row_end : c->N};
  if (g.row_end <= g.row_beg) return;                       // this rank owns no rows (more ranks than tile rows)
  if (c->use_tma && c->N > GEMM_SMALL_N) {
    const CUtensorMap& mA0 = nn_map(c, A0);
    const CUtensorMap& mB0 = nn_map(c, B0);
    const int2* tiles = c->d_tiles_sym;
    int ntiles = c->pp.T;
    if (shard) { sym = 0; tiles = c->d_tiles_full + (size_t)(c->row_beg / TILE) * c->ntile; ntiles = ((c->row_end - c->row_beg + TILE - 1) / TILE) * c->ntile; }
    else if (!sym) { tiles = c->d_tiles_full; ntiles = c->ntile * c->ntile; }
    launch_gemm_abt_tma(g, mA0, mB0, A1 ? nn_map(c, A1) : mA0, B1 ? nn_map(c, B1) : mB0, sym, tiles, ntiles, c->gemm_ws,
                        c->gemm_sync, c->sms, c->st);
  } else {
    launch_gemm_abt(g, c->st);
  }
  c->launches += 1;
}

// C = cos X, S = sin X for the real symmetric X (H-bar real at Gamma) -> U = C - i S.
// cos X = sum_k (-1)^k Y^k/(2k)!, sin X = X sum_k (-1)^k Y^k/(2k+1)!, Y = X^2, k <= q.   q + 1 GEMMs.
// With the powers Y^2 .. Y^q kept (Yb, Yc and q - 3 more matrices, allocated when they fit) the products carry no
// read-modify-write of C and Sc in their epilogues -- those ran the DMMA pipe at 70 % against 91 % for the plain product
// (ncu, N = 2,400) -- and one elementwise kernel sums the two series afterwards, in the same order.
void enqueue_expm(rt_ctx* c) {
  if (c->q >= 2 && (int)c->pw_extra.size() >= c->q - 3 && c->q <= SERIES_MAX_Q) {
    enqueue_gemm(c, 1, c->X, c->X, 1.0, nullptr, nullptr, 0, c->Ya);
    SeriesArgs sa{};
    sa.q = c->q;
    sa.pw[0] = c->Ya;
    sa.c[0] = -0.5; sa.s[0] = -1.0 / 6.0;
    const double* prev = c->Ya;
    for (int k = 2; k <= c->q; ++k) {
      sa.c[k - 1] = -sa.c[k - 2] / ((2.0 * k - 1.0) * (2.0 * k));
      sa.s[k - 1] = -sa.s[k - 2] / ((2.0 * k) * (2.0 * k + 1.0));
      double* cur = k == 2 ? c->Yb : (k == 3 ? c->Yc : c->pw_extra[k - 4]);
      enqueue_gemm(c, 1, prev, c->Ya, 1.0, nullptr, nullptr, 0, cur);
      sa.pw[k - 1] = cur;
      prev = cur;
    }
    launch_series_combine(c->N, c->ldn, sa, c->Cm, c->Sc, 0, c->N, c->st);
    c->launches += 1;
    enqueue_gemm(c, 1, c->X, c->Sc, 1.0, nullptr, nullptr, 0, c->Sm);
    return;
  }
  enqueue_gemm(c, 1, c->X, c->X, 1.0, nullptr, nullptr, 0, c->Ya);
  launch_series_init(c->N, c->ldn, c->Ya, c->Cm, -0.5, c->Sc, -1.0 / 6.0, c->st);
  c->launches += 1;
  double ck = -0.5, sk = -1.0 / 6.0;
  const double* prev = c->Ya;
  for (int k = 2; k <= c->q; ++k) {
    ck = -ck / ((2.0 * k - 1.0) * (2.0 * k));
    sk = -sk / ((2.0 * k) * (2.0 * k + 1.0));
    double* cur = (k < c->q) ? ((k & 1) ? c->Yc : c->Yb) : nullptr;
    enqueue_gemm(c, 1, prev, c->Ya, 1.0, nullptr, nullptr, 0, cur, c->Cm, ck, c->Sc, sk);
    prev = cur;
  }
  enqueue_gemm(c, 1, c->X, c->Sc, 1.0, nullptr, nullptr, 0, c->Sm);
}

// P1 = U P0 U^dagger (Eq. 15), U = C - iS, P0 = A + iB (A symmetric, B antisymmetric).
//   Yr = C A + S B, Yi = C B - S A ; P1r = Yr C - Yi S, P1i = Yr S + Yi C.
// gemm_abt contracts against B^T: a symmetric right factor is used as is, the antisymmetric one flips the sign.
// need_im = false: Im P1 is not formed.  Only the LAST Hamiltonian update of a step hands its P1 on (line 28); the earlier
// ones are read by the density alone, which takes Re P1 (Eq. 27: Im P is antisymmetric and drops out for real orbitals).
void enqueue_upu(rt_ctx* c, const double* Ar, const double* Ai, double* Or, double* Oi, bool need_im = true) {
  enqueue_gemm(c, 0, c->Cm, Ar, 1.0, c->Sm, Ai, -1.0, c->Yb);
  enqueue_gemm(c, 0, c->Cm, Ai, -1.0, c->Sm, Ar, -1.0, c->Yc);
  enqueue_gemm(c, 1, c->Yb, c->Cm, 1.0, c->Yc, c->Sm, -1.0, Or);      // P1 Hermitian: Re symmetric,
  if (need_im) enqueue_gemm(c, -1, c->Yb, c->Sm, 1.0, c->Yc, c->Cm, 1.0, Oi);      // Im antisymmetric
}

// ---- the same propagation with the N^3 work sharded over ranks by row blocks ("once N exceeds a few
// thousands" the multi-GPU product wins over the replicated one).  D = A B^T needs only the rows of A that the rank
// owns and all of B, so a chain prev -> prev * Y stays local; three points need a matrix complete on every rank, and
// the caller all-gathers the row blocks there (rt_slab_get_shard):
//   A: Y = X X^T                                                        -> gather Y
//   B: powers of Y, C = cos X, Sc = sinc-series, S = Sc X, Yr, Yi        -> gather C, S   (right factors of the last two)
//   C: P1r = Yr C - Yi S, P1i = Yr S + Yi C                              -> gather P1r, P1i
//   D: P1 made exactly Hermitian from its upper triangle (both triangles were computed separately), then the density
// Every element is computed by exactly one rank, so all ranks hold bit-identical matrices after each gather.
void enqueue_shard_A(rt_ctx* c, int it) {
  stage_begin(c, RT_STAGE_ELDYN);
  if (c->d_cs) cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st);
  launch_hbar(c->N, c->ldn, c->Hm1, c->H0, c->H1, c->X, c->dt, c->sigma, it == 0, c->st);       // lines 11, 14 (replicated)
  c->launches += 1;
  enqueue_gemm(c, 0, c->X, c->X, 1.0, nullptr, nullptr, 0, c->Ya, nullptr, 0, nullptr, 0, nullptr, true);
  stage_end(c);
}
void enqueue_shard_B(rt_ctx* c) {
  stage_begin(c, RT_STAGE_ELDYN);
  if (c->q >= 2 && (int)c->pw_extra.size() >= c->q - 3 && c->q <= SERIES_MAX_Q) {
    // stored powers (see enqueue_expm): the rank's row block of every power, then the series on those rows
    SeriesArgs sa{};
    sa.q = c->q;
    sa.pw[0] = c->Ya;
    sa.c[0] = -0.5; sa.s[0] = -1.0 / 6.0;
    const double* prev = c->Ya;
    for (int k = 2; k <= c->q; ++k) {
      sa.c[k - 1] = -sa.c[k - 2] / ((2.0 * k - 1.0) * (2.0 * k));
      sa.s[k - 1] = -sa.s[k - 2] / ((2.0 * k) * (2.0 * k + 1.0));
      double* cur = k == 2 ? c->Yb : (k == 3 ? c->Yc : c->pw_extra[k - 4]);
      enqueue_gemm(c, 0, prev, c->Ya, 1.0, nullptr, nullptr, 0, cur, nullptr, 0, nullptr, 0, nullptr, true);
      sa.pw[k - 1] = cur;
      prev = cur;
    }
    launch_series_combine(c->N, c->ldn, sa, c->Cm, c->Sc, c->row_beg, c->row_end, c->st);
    c->launches += 1;
    enqueue_gemm(c, 0, c->Sc, c->X, 1.0, nullptr, nullptr, 0, c->Sm, nullptr, 0, nullptr, 0, nullptr, true);   // S = Sc X (commute)
    enqueue_gemm(c, 0, c->Cm, c->P0r, 1.0, c->Sm, c->P0i, -1.0, c->Yb, nullptr, 0, nullptr, 0, nullptr, true);
    enqueue_gemm(c, 0, c->Cm, c->P0i, -1.0, c->Sm, c->P0r, -1.0, c->Yc, nullptr, 0, nullptr, 0, nullptr, true);
    stage_end(c);
    return;
  }
  launch_series_init(c->N, c->ldn, c->Ya, c->Cm, -0.5, c->Sc, -1.0 / 6.0, c->st);    // elementwise on the whole matrix
  c->launches += 1;
  double ck = -0.5, sk = -1.0 / 6.0;
  const double* prev = c->Ya;
  for (int k = 2; k <= c->q; ++k) {
    ck = -ck / ((2.0 * k - 1.0) * (2.0 * k));
    sk = -sk / ((2.0 * k) * (2.0 * k + 1.0));
    double* cur = (k < c->q) ? ((k & 1) ? c->Yc : c->Yb) : nullptr;
    enqueue_gemm(c, 0, prev, c->Ya, 1.0, nullptr, nullptr, 0, cur, c->Cm, ck, c->Sc, sk, nullptr, true);
    prev = cur;
  }
  enqueue_gemm(c, 0, c->Sc, c->X, 1.0, nullptr, nullptr, 0, c->Sm, nullptr, 0, nullptr, 0, nullptr, true);   // S = Sc X (commute)
  enqueue_gemm(c, 0, c->Cm, c->P0r, 1.0, c->Sm, c->P0i, -1.0, c->Yb, nullptr, 0, nullptr, 0, nullptr, true);
  enqueue_gemm(c, 0, c->Cm, c->P0i, -1.0, c->Sm, c->P0r, -1.0, c->Yc, nullptr, 0, nullptr, 0, nullptr, true);
  stage_end(c);
}
void enqueue_shard_C(rt_ctx* c) {
  stage_begin(c, RT_STAGE_ELDYN);
  enqueue_gemm(c, 0, c->Yb, c->Cm, 1.0, c->Yc, c->Sm, -1.0, c->P1r, nullptr, 0, nullptr, 0, nullptr, true);
  // (Im P1 is formed and gathered on every update here: the caller's gather list is fixed per phase)
  enqueue_gemm(c, 0, c->Yb, c->Sm, 1.0, c->Yc, c->Cm, 1.0, c->P1i, nullptr, 0, nullptr, 0, nullptr, true);
  stage_end(c);
}

// The paper's propagator (Eq. 39, Alg. 1 lines 15-23 L375-L392) with S = 1 and Hbar real symmetric (L433):
//   dP^(k) = (1/k)(Omega dP^(k-1) + dP^(k-1) Omega^dagger) = (-i/k)[X, dP^(k-1)],  X = dt Hbar;  P1 = P0 + sum_k dP^(k)
// split as in Eq. 40 (L428-L433) with dP = S' + iA':   S'' = (1/k)[X, A'],  A'' = -(1/k)[X, S'].
// Each commutator is ONE dual-term GEMM whose output is known to be (anti)symmetric, so only the upper tiles are
// computed and mirrored -- the same 2N^3 flop as the paper's "one multiply + transpose (DGEAM)" form (L434-L438).
// gemm_abt contracts against B^T:  X A' = -gemm(X, A'),  A' X = gemm(A', X),  X S' = gemm(X, S'),  S' X = gemm(S', X).
// (X carries the shift -sigma dt I, which commutes with everything.)  The loop `while dP_err > dP_thrs` runs on the
// device: commutator_check sets cs->done and the GEMMs of the remaining orders (up to kmax) return immediately.
void enqueue_commutator(rt_ctx* c, const double* Ar, const double* Ai, double* Or, double* Oi) {
  const size_t nn = (size_t)c->N * c->ldn * 8;
  cudaMemcpyAsync(Or, Ar, nn, cudaMemcpyDeviceToDevice, c->st);               // line 15: P1 <- P0
  cudaMemcpyAsync(Oi, Ai, nn, cudaMemcpyDeviceToDevice, c->st);
  const double* pr = Ar;                                                      // line 17 (DESIGN R2): dP <- P0
  const double* pi = Ai;
  double* bufs[2][2] = {{c->Yb, c->Yc}, {c->Cm, c->Sm}};
  const int* skip = &c->d_cs->done;
  for (int k = 1; k <= c->kmax; ++k) {
    double* nr = bufs[k & 1][0];
    double* ni = bufs[k & 1][1];
    const double s = 1.0 / (double)k;
    enqueue_gemm(c, 1, c->X, pi, -s, pi, c->X, -s, nr, Or, 1.0, nullptr, 0, skip);    // S'' and P1r += S''  (lines 20-21)
    enqueue_gemm(c, -1, c->X, pr, -s, pr, c->X, s, ni, Oi, 1.0, nullptr, 0, skip);    // A'' and P1i += A''
    launch_commutator_check(c->N, c->ldn, nr, ni, k, c->dP_thrs, c->d_cs, c->st);     // line 22
    c->launches += 1;
    pr = nr;
    pi = ni;
  }
}

// The same series for a GENERAL Omega = -i B + W (Eq. 21-23; Eq. 37-38):
//   B = dt (S^-1 Hbar - sigma 1)      real, symmetric only when S = 1        (Eq. 36; the shift commutes)
//   W = dt^2/12 [S^-1 H0, S^-1 H1]    real, second Magnus term (Eq. 13); absent for magnus = 1
//   dP^(k) = (1/k)(Omega dP + dP Omega^dagger) = (1/k)(M + M^dagger),  M = Omega dP^(k-1),  dP = S' + i A':
//   Re M = B A' + W S',  Im M = -B S' + W A'  ->  S'' = (Re M + Re M^T)/k,  A'' = (Im M - Im M^T)/k.
// This is the paper's "one matrix-matrix multiplication and a matrix transpose (DGEAM)" form (L434-L438): two full
// (dual-term) GEMMs and one transpose-add kernel per order.  gemm_abt contracts against the second operand transposed:
// B A' = -gemm(B, A'), W S' = gemm(W, S'), B S' = gemm(B, S'), W A' = -gemm(W, A').
void enqueue_general_omega(rt_ctx* c) {
  const double* X = c->X;                               // dt (Hbar - sigma S) from launch_hbar
  if (c->nonorth) {
    enqueue_gemm(c, 0, c->Sinv, X, 1.0, nullptr, nullptr, 0, c->Bm);                    // B = S^-1 X  (X symmetric)
  }
  if (c->magnus >= 2) {
    const double w12 = c->dt * c->dt / 12.0;
    if (!c->nonorth) {
      enqueue_gemm(c, -1, c->H0, c->H1, w12, c->H1, c->H0, -w12, c->Wm);                // dt^2/12 (H0 H1 - H1 H0)
    } else {
      // G_a = S^-1 H_a and G_a^T = H_a S^-1 in the (still free) series buffers, then W = dt^2/12 (G0 G1 - G1 G0)
      enqueue_gemm(c, 0, c->Sinv, c->H0, 1.0, nullptr, nullptr, 0, c->Yb);              // G0
      enqueue_gemm(c, 0, c->Sinv, c->H1, 1.0, nullptr, nullptr, 0, c->Yc);              // G1
      enqueue_gemm(c, 0, c->H0, c->Sinv, 1.0, nullptr, nullptr, 0, c->Cm);              // G0^T
      enqueue_gemm(c, 0, c->H1, c->Sinv, 1.0, nullptr, nullptr, 0, c->Sm);              // G1^T
      enqueue_gemm(c, 0, c->Yb, c->Sm, w12, c->Yc, c->Cm, -w12, c->Wm);
    }
  }
}

void enqueue_commutator_general(rt_ctx* c, const double* Ar, const double* Ai, double* Or, double* Oi) {
  const size_t nn = (size_t)c->N * c->ldn * 8;
  enqueue_general_omega(c);
  cudaMemcpyAsync(Or, Ar, nn, cudaMemcpyDeviceToDevice, c->st);               // P1 <- P0
  cudaMemcpyAsync(Oi, Ai, nn, cudaMemcpyDeviceToDevice, c->st);
  const double* B = c->nonorth ? c->Bm : c->X;
  const double* W = c->magnus >= 2 ? c->Wm : nullptr;
  const double* pr = Ar;
  const double* pi = Ai;
  double* bufs[2][2] = {{c->Yb, c->Yc}, {c->Cm, c->Sm}};
  const int* skip = &c->d_cs->done;
  for (int k = 1; k <= c->kmax; ++k) {
    double* nr = bufs[k & 1][0];
    double* ni = bufs[k & 1][1];
    if (W) {
      enqueue_gemm(c, 0, B, pi, -1.0, W, pr, 1.0, c->Rt, nullptr, 0, nullptr, 0, skip);      // Re M
      enqueue_gemm(c, 0, B, pr, -1.0, W, pi, -1.0, c->It, nullptr, 0, nullptr, 0, skip);     // Im M
    } else {
      enqueue_gemm(c, 0, B, pi, -1.0, nullptr, nullptr, 0, c->Rt, nullptr, 0, nullptr, 0, skip);
      enqueue_gemm(c, 0, B, pr, -1.0, nullptr, nullptr, 0, c->It, nullptr, 0, nullptr, 0, skip);
    }
    launch_transpose_add(c->N, c->ldn, c->Rt, c->It, 1.0 / (double)k, nr, ni, Or, Oi, skip, c->st);
    launch_commutator_check(c->N, c->ldn, nr, ni, k, c->dP_thrs, c->d_cs, c->st);             // line 22
    c->launches += 2;
    pr = nr;
    pi = ni;
  }
}

void enqueue_propagate(rt_ctx* c, const double* Ar, const double* Ai, double* Or, double* Oi, bool need_im = true) {
  if (c->general) enqueue_commutator_general(c, Ar, Ai, Or, Oi);
  else if (c->prop == RT_PROP_COMMUTATOR) enqueue_commutator(c, Ar, Ai, Or, Oi);
  else { enqueue_expm(c); enqueue_upu(c, Ar, Ai, Or, Oi, need_im); }
}

void enqueue_density(rt_ctx* c, const double* reP, double* rho_out, const double* rho0) {
  launch_fold_upper(c->N, c->ldn, reP, c->X, c->st);
  if (c->use_tma)
    launch_density_tma(c->dp, nn_map(c, c->X), c->tmPhiN, c->phiN_3d, c->phi, c->d_segs, c->rho_part, c->sms,
                       c->dens_resident ? nullptr : c->pace_cnt, c->pace_w, c->dens_resident ? 1 : 0, c->st);
  else launch_density(c->dp, c->phi, c->X, c->rho_part, c->st);
  launch_reduce_rho(c->rho_part, c->use_tma ? c->dp.ntypes : c->dp.npairs, c->Ngl, c->gd, c->h, c->x0, rho0, rho_out,
                    c->d_bsums, c->d_sums, c->st);
  c->launches += 4;
}

// a7: one Poisson solve on the hierarchy `lv` (lv[0].u is warm-started), right-hand side from rho - rho0
void enqueue_poisson(rt_ctx* c, const std::vector<MgLevel>& lv, int n_vc, const double* rho, const double* rho0) {
  MgSolveArgs s{lv.data(), (int)lv.size(), n_vc, c->nu1, c->nu2, c->omega, c->Qx, c->Qy, c->Qz, c->lx, c->ly, c->lz,
                rho, rho0, c->d_sums};
  if (c->fd_order == 4) c->launches += launch_mg_solve_order4(s, c->dl0, c->f4, c->st);   // 13-point operator, MG-preconditioned
  else c->launches += launch_mg_solve(s, c->st);
}

// v_xc(rho) into out (LDA: one elementwise kernel; PBE: gradient pass + divergence pass)
void enqueue_vxc(rt_ctx* c, const double* rho, double* out) {
  if (c->xc_kind == RT_XC_PBE) {
    launch_vxc_pbe(c->gd, c->h, c->fd_order, rho, c->pbe_scr, out, nullptr, c->st);
    c->launches += 2;
  } else {
    launch_vxc(c->Ng, rho, out, c->st);
    c->launches += 1;
  }
}

// eps != nullptr: the ground-state Hamiltonian is added -- diag(eps), or the matrix Hks of rt_create_general
void enqueue_project(rt_ctx* c, const double* w, const double* eps, double* H) {
  if (c->use_tma) launch_project_tma(c->pp, c->tmPhiK, w, c->d_tiles, c->W, c->sms, c->pace_cnt, c->pace_w, c->st);
  else launch_project(c->pp, c->phi, w, c->d_tiles, c->W, c->st);
  const bool mat = eps && c->Hks;
  launch_project_reduce(c->pp, c->W, mat ? nullptr : eps, c->dvol, H, c->st, mat ? c->Hks : nullptr);
  c->launches += 2;
}

// H = diag(eps) + dVol Phi diag(w) Phi^T with w = c->w (whole grid).  A slab handle contracts over its own grid
// points only (the partial sum of PAPER.md:L424; the slab of w is first copied to the 16-byte aligned op_u) and only
// the rank that owns plane 0 adds diag(eps), so that the all-reduce of the partial matrices gives H.
void enqueue_project_dv(rt_ctx* c, double* H) {
  if (!c->slab) { enqueue_project(c, c->w, c->d_eps, H); return; }
  cudaMemcpyAsync(c->op_u, c->w + c->slab_off, (size_t)c->Ngl * 8, cudaMemcpyDeviceToDevice, c->st);
  enqueue_project(c, c->op_u, c->x0 == 0 ? c->d_eps : nullptr, H);
}

void enqueue_density_stage(rt_ctx* c) {
  stage_begin(c, RT_STAGE_RHO);
  if (c->slab) cudaMemsetAsync(c->rho, 0, (size_t)(c->Ng + 8) * 8, c->st);                     // other ranks' slabs
  enqueue_density(c, c->P1r, c->rho + c->slab_off, c->rho0 + c->slab_off);                     // Eq. 27 + line 27
  stage_end(c);
}

// First half of a Hamiltonian update, Algorithm 1 lines 14-23 + Eq. 27 (`it` = 0 also extrapolates H1, line 11):
// mean Hamiltonian, propagation, density of this handle's grid points (+ partial dipole / charge sums).
void enqueue_update_propagate(rt_ctx* c, int it) {
  stage_begin(c, RT_STAGE_ELDYN);
  if (c->d_cs) cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st);                          // lines 12, 16
  launch_hbar(c->N, c->ldn, c->Hm1, c->H0, c->H1, c->X, c->dt, c->sigma, it == 0, c->st, c->Smat);   // lines 11, 14
  c->launches += 1;
  // fixed-count step: only the last update's Im P1 is ever read (by line 28); the dynamic loop cannot know which is last
  const bool need_im = c->dynamic || it >= c->m - 1;
  enqueue_propagate(c, c->P0r, c->P0i, c->P1r, c->P1i, need_im);                               // Eq. 15 / Eq. 39
  stage_end(c);
  enqueue_density_stage(c);
}

// Second half, lines 24-25: potential update on the whole grid from the (complete) density, then the projection
// over this handle's grid points.
void enqueue_update_potential(rt_ctx* c) {
  if (c->use_h) {
    stage_begin(c, RT_STAGE_VH);
    enqueue_poisson(c, c->lv, c->n_vc, c->rho, c->rho0);
    stage_end(c);
  }

  stage_begin(c, RT_STAGE_XC);
  if (c->xc_kind == RT_XC_PBE && c->use_xc) {
    enqueue_vxc(c, c->rho, c->vxc_cur);
    launch_delta_v_assemble(c->Ng, c->gd, c->h, c->vxc_cur, c->vxc0, c->use_h ? c->lv[0].u : nullptr, c->d_E, c->w, c->st);
  } else {
    launch_delta_v(c->Ng, c->gd, c->h, c->rho, c->vxc0, c->lv[0].u, c->d_E, c->use_h, c->use_xc, c->w, c->st);
  }
  c->launches += 1;
  stage_end(c);

  stage_begin(c, RT_STAGE_HUPDATE);
  if (c->dynamic)                                                                              // H1_old <- H1
    cudaMemcpyAsync(c->Ya, c->H1, (size_t)c->N * c->ldn * 8, cudaMemcpyDeviceToDevice, c->st);
  enqueue_project_dv(c, c->H1);                                                                // line 25
  if (c->dynamic && !c->slab) {               // a slab holds a partial sum here: RT_SLAB_CHECK measures after the all-reduce
    launch_maxabs_diff(c->N, c->ldn, c->H1, c->Ya, c->d_cs, c->st);                            // line 24
    c->launches += 1;
  }
  stage_end(c);
}

void enqueue_update(rt_ctx* c, int it) {
  enqueue_update_propagate(c, it);
  enqueue_update_potential(c);
}

void enqueue_record(rt_ctx* c) {                 // Alg. 1 line 27: the dipole of this time level joins the series
  if (!c->hist_cap) return;
  launch_record_dipole(c->d_sums, c->dvol, c->d_hist, c->hist_cap, c->d_hist_n, c->st);
  c->launches += 1;
}

void enqueue_shift(rt_ctx* c) {
  launch_copy5(c->N, c->ldn, c->Hm1, c->H0, c->H0, c->H1, c->P0r, c->P1r, c->P0i, c->P1i, c->st);   // line 28
  c->launches += 1;
  enqueue_record(c);
}

// One time step with a fixed number of Hamiltonian updates, Algorithm 1 lines 10-28.
void enqueue_step(rt_ctx* c) {
  for (int it = 0; it < c->m; ++it) enqueue_update(c, it);
  enqueue_shift(c);
}

int sync_and_check(rt_ctx* c) {
  CK(cudaStreamSynchronize(c->st));
  CK(cudaGetLastError());
  return RT_OK;
}

int collect_timing(rt_ctx* c) {
  for (auto& ep : c->ev_used) {
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, ep.a, ep.b));
    c->stage_ms[ep.stage] += ms;
    c->stage_calls[ep.stage] += 1;
    c->ev_free.push_back(ep);
  }
  c->ev_used.clear();
  return RT_OK;
}

int copy_matrix_out(rt_ctx* c, const double* src, double* dst) {   // [N][ldn] device -> [N][N] anywhere
  if (!dst) return RT_OK;
  CK(cudaMemcpy2DAsync(dst, (size_t)c->N * 8, src, (size_t)c->ldn * 8, (size_t)c->N * 8, c->N, cudaMemcpyDefault, c->st));
  return RT_OK;
}
int copy_matrix_in(rt_ctx* c, const double* src, double* dst) {    // [N][N] anywhere -> [N][ldn] device
  CK(cudaMemsetAsync(dst, 0, (size_t)c->N * c->ldn * 8, c->st));
  CK(cudaMemcpy2DAsync(dst, (size_t)c->ldn * 8, src, (size_t)c->N * 8, (size_t)c->N * 8, c->N, cudaMemcpyDefault, c->st));
  return RT_OK;
}

}  // namespace

// ======================================================================================================
extern "C" {

const char* rt_last_error(rt_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int rt_destroy(rt_handle c) {
  if (!c) return RT_OK;
  cudaSetDevice(c->cfg.device);
  cudaStreamSynchronize(c->st);
  if (c->gexec) cudaGraphExecDestroy(c->gexec);
  if (c->graph) cudaGraphDestroy(c->graph);
  for (int i = 0; i < 2; ++i) {
    if (c->gexec_upd[i]) cudaGraphExecDestroy(c->gexec_upd[i]);
    if (c->graph_upd[i]) cudaGraphDestroy(c->graph_upd[i]);
  }
  for (auto& kv : c->phase_exec) cudaGraphExecDestroy(kv.second);
  for (auto g : c->phase_graphs) cudaGraphDestroy(g);
  for (auto& ep : c->ev_used) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  for (auto& ep : c->ev_free) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  for (void* p : c->allocs) cudaFree(p);
  cudaGetLastError();
  delete c;
  return RT_OK;
}

}  // extern "C"

namespace {
// Common body of rt_create (Hks = P0re = P0im = nullptr: KS basis, H_KS = diag(eps), P0 = diag(occ)) and
// rt_create_general (ground state given as matrices; occ may be nullptr).
int create_impl(const rt_config* cfg, const double* phi, const double* eps, const double* occ, const double* Hks_in,
                const double* P0re_in, const double* P0im_in, rt_handle* out) {
  rt_ctx* c = nullptr;
  if (!cfg || !phi || !eps || !out || (!occ && !P0re_in)) return fail(c, RT_EINVAL, "rt_create: NULL argument");
  *out = nullptr;
  const bool want_nonorth = (cfg->flags & RT_NONORTHOGONAL) != 0;
  const bool want_general = want_nonorth || cfg->magnus_order >= 2;
  if (cfg->magnus_order < 0 || cfg->magnus_order > 2) return fail(c, RT_EINVAL, "rt_create: magnus_order must be 0, 1 or 2");
  if (want_general && cfg->propagator != RT_PROP_COMMUTATOR)
    return fail(c, RT_EINVAL, "rt_create: the second Magnus term and a non-orthogonal basis are propagated with the paper's "
                              "series (Eq. 37-38): set propagator = RT_PROP_COMMUTATOR");
  if (want_general && cfg->slab_nx > 0)
    return fail(c, RT_EINVAL, "rt_create: magnus_order = 2 / RT_NONORTHOGONAL are not available on slab handles");
  if (cfg->xc_functional != RT_XC_LDA_PZ81 && cfg->xc_functional != RT_XC_PBE)
    return fail(c, RT_EINVAL, "rt_create: unknown xc_functional");
  if (cfg->fd_order != 0 && cfg->fd_order != 2 && cfg->fd_order != 4)
    return fail(c, RT_EINVAL, "rt_create: fd_order must be 0, 2 or 4");
  if (want_nonorth && !(Hks_in && P0re_in))
    return fail(c, RT_EINVAL, "rt_create: RT_NONORTHOGONAL needs the ground state as matrices (rt_create_general)");
  if (cfg->nx < 2 || cfg->ny < 2 || cfg->nz < 2) return fail(c, RT_EINVAL, "rt_create: grid dims must be >= 2");
  if (!(cfg->h > 0) || !(cfg->dt > 0)) return fail(c, RT_EINVAL, "rt_create: h and dt must be > 0");
  if (cfg->norb < 1) return fail(c, RT_EINVAL, "rt_create: norb must be >= 1");
  if (cfg->n_hupdates < 0 || cfg->n_vcycles < 0 || cfg->nu_pre < 0 || cfg->nu_post < 0 || cfg->exp_order < 0)
    return fail(c, RT_EINVAL, "rt_create: negative iteration count");
  if (cfg->propagator != RT_PROP_TAYLOR && cfg->propagator != RT_PROP_COMMUTATOR)
    return fail(c, RT_EINVAL, "rt_create: unknown propagator");
  if (cfg->slab_nx < 0 || cfg->slab_x0 < 0 || (cfg->slab_nx > 0 && cfg->slab_x0 + cfg->slab_nx > cfg->nx))
    return fail(c, RT_EINVAL, "rt_create: slab [slab_x0, slab_x0 + slab_nx) must lie inside [0, nx)");
  if (cfg->prop_shards < 0 || (cfg->prop_shards > 1 && (cfg->prop_shard < 0 || cfg->prop_shard >= cfg->prop_shards)))
    return fail(c, RT_EINVAL, "rt_create: prop_shard must lie in [0, prop_shards)");
  if (cfg->prop_shards > 1 && cfg->slab_nx == 0)
    return fail(c, RT_EINVAL, "rt_create: the row-sharded propagator is part of the slab protocol (set slab_nx)");
  if (cfg->prop_shards > 1 && cfg->propagator != RT_PROP_TAYLOR)
    return fail(c, RT_EINVAL, "rt_create: the row-sharded propagator implements the Taylor mode only");
  if (cfg->history < 0) return fail(c, RT_EINVAL, "rt_create: history < 0");
  if (cfg->max_order < 0 || cfg->max_order > MAX_ORDER || cfg->max_hupdates < 0 || !(cfg->dP_thrs >= 0.0) ||
      !(cfg->H_thrs >= 0.0))
    return fail(c, RT_EINVAL, "rt_create: bad max_order / max_hupdates / dP_thrs / H_thrs");
  for (int i = 0; occ && i < cfg->norb; ++i)
    if (!(occ[i] >= 0.0 && occ[i] <= 2.0)) return fail(c, RT_EINVAL, "rt_create: occ must lie in [0, 2]");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) {
    cudaGetLastError();
    return fail(c, RT_ECUDA, "rt_create: no such CUDA device (this library has no CPU fallback)");
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess || prop.major < 10)
    return fail(c, RT_ECUDA, "rt_create: device is not sm_100 or newer");
  if (cudaSetDevice(cfg->device) != cudaSuccess) return fail(c, RT_ECUDA, "rt_create: cudaSetDevice failed");

  c = new rt_ctx();
  c->cfg = *cfg;
  c->N = cfg->norb;
  c->ldn = roundup(c->N, 8);
  c->ntile = (c->N + TILE - 1) / TILE;
  c->nshard = cfg->prop_shards > 1 ? cfg->prop_shards : 1;
  c->shard = c->nshard > 1 ? cfg->prop_shard : 0;
  c->shard_rows = ((c->ntile + c->nshard - 1) / c->nshard) * TILE;       // whole tile rows per rank
  c->row_beg = std::min(c->N, c->shard * c->shard_rows);
  c->row_end = std::min(c->N, (c->shard + 1) * c->shard_rows);
  c->nn_alloc = (size_t)std::max(c->N, c->nshard * c->shard_rows) * c->ldn;
  c->gd = GridDims{cfg->nx, cfg->ny, cfg->nz};
  c->Ng = (long long)cfg->nx * cfg->ny * cfg->nz;
  c->Ngl = c->Ng;
  if (cfg->slab_nx > 0) {
    c->slab = true;
    c->x0 = cfg->slab_x0;
    c->Ngl = (long long)cfg->slab_nx * cfg->ny * cfg->nz;
    c->slab_off = (long long)cfg->slab_x0 * cfg->ny * cfg->nz;
  }
  c->h = cfg->h;
  c->dvol = cfg->h * cfg->h * cfg->h;
  c->dt = cfg->dt;
  c->m = cfg->n_hupdates ? cfg->n_hupdates : 2;
  c->n_vc = cfg->n_vcycles;
  c->nu1 = (cfg->nu_pre || cfg->nu_post) ? cfg->nu_pre : 2;
  c->nu2 = (cfg->nu_pre || cfg->nu_post) ? cfg->nu_post : 2;
  c->omega = cfg->jacobi_omega != 0.0 ? cfg->jacobi_omega : 6.0 / 7.0;
  c->use_h = !(cfg->flags & RT_NO_HARTREE);
  c->use_xc = !(cfg->flags & RT_NO_XC);
  c->use_graph = !(cfg->flags & RT_NO_GRAPH);
  c->xc_kind = cfg->xc_functional;
  c->fd_order = cfg->fd_order == 4 ? 4 : 2;
  c->magnus = cfg->magnus_order >= 2 ? 2 : 1;
  c->nonorth = want_nonorth;
  c->general = want_general;
  c->st = reinterpret_cast<cudaStream_t>(cfg->stream);
  const int N = c->N, ldn = c->ldn;
  const long long Ng = c->Ngl;      // grid points of this handle's Phi: what the plans and Phi descriptors see
  const long long NgF = c->Ng;      // the whole grid: every O(Ng) array and the Poisson / xc stages

#define FAIL_CREATE(code, msg) do { int rc_ = fail(nullptr, (code), (msg)); rt_destroy(c); return rc_; } while (0)
#define CKC(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { std::string m_ = std::string(#call) + ": " + cudaGetErrorString(e_); cudaGetLastError(); FAIL_CREATE(RT_ECUDA, m_); } } while (0)
#define ALLOC(ptr, count) do { if (dev_alloc(c, &(ptr), (size_t)(count)) != RT_OK) { std::string m_ = c->err; FAIL_CREATE(RT_ENOMEM, m_); } } while (0)

  // series order from the spectral bound (DESIGN R8)
  double emin = eps[0], emax = eps[0];
  for (int i = 1; i < N; ++i) { emin = std::fmin(emin, eps[i]); emax = std::fmax(emax, eps[i]); }
  c->sigma = 0.5 * (emin + emax);
  {
    const double half[3] = {0.5 * (cfg->nx - 1) * cfg->h, 0.5 * (cfg->ny - 1) * cfg->h, 0.5 * (cfg->nz - 1) * cfg->h};
    double vmax = 0.5;
    for (int d = 0; d < 3; ++d) vmax += std::fabs(cfg->E0[d]) * half[d];
    const double theta = c->dt * (0.5 * (emax - emin) + vmax);
    c->theta0 = c->dt * (0.5 * (emax - emin) + 0.5);
    for (int d = 0; d < 3; ++d) c->half_len[d] = half[d];
    int q;
    if (cfg->exp_order > 0) q = (cfg->exp_order > 1) ? cfg->exp_order / 2 : 1;   // degree 2q+1 >= K
    else {
      q = 1;
      double term = theta * theta * theta * theta / 24.0;     // theta^(2q+2)/(2q+2)! at q = 1
      while (term > 1e-17 && q < 40) { ++q; term *= theta * theta / ((2.0 * q + 1.0) * (2.0 * q + 2.0)); }
    }
    c->q = q;
    // the paper's loops: thresholds of Alg. 1 line 5 (L351); kmax from the same spectral bound -- the k-th term of
    // the commutator series is bounded by max|P0| (2 theta)^k / k!  (||ad_X|| <= 2 ||X||)
    c->prop = cfg->propagator;
    c->dP_thrs = cfg->dP_thrs > 0.0 ? cfg->dP_thrs : 1e-10;
    c->H_thrs = cfg->H_thrs;
    c->dynamic = cfg->H_thrs > 0.0;
    c->max_hup = cfg->max_hupdates > 0 ? cfg->max_hupdates : 20;
    if (cfg->max_order > 0) c->kmax = cfg->max_order;
    else {
      int k = 1;
      double term = 2.0 * 2.0 * theta;
      while (term > 1e-3 * c->dP_thrs && k < MAX_ORDER) { ++k; term *= 2.0 * theta / k; }
      c->kmax = k + 2 < MAX_ORDER ? k + 2 : MAX_ORDER;
    }
  }

  // multigrid hierarchy
  {
    GridDims g = c->gd;
    double hh = c->h;
    for (;;) {
      MgLevel L{};
      L.gd = g; L.h = hh; L.n = (long long)g.nx * g.ny * g.nz;
      c->lv.push_back(L);
      if (!can_coarsen(g)) break;
      g = GridDims{g.nx / 2, g.ny / 2, g.nz / 2};
      hh *= 2.0;
    }
    // a coarsest level of any size is accepted: beyond 32768 points its exact separable solve runs as six whole-GPU
    // launches (mg_kernels.cu launch_coarse_exact_global); the eigenvector tables below are then up to ~10^5 doubles
  }

  // plans
  const int ntile = (N + TILE - 1) / TILE;
  {
    ProjectPlan& p = c->pp;
    p.N = N; p.Ng = Ng; p.ntile = ntile; p.T = ntile * (ntile + 1) / 2; p.ldn = ldn;
    // Split-K factors.  One CTA per SM, CTAs handed out in block order: the plan is the (S, Sn, Sd) whose greedy
    // schedule on `sms` machines finishes first.  Cost model in pipeline stages (16 grid points of one 128 x 128 tile): a
    // full CTA costs kchunk/16, a narrow one 0.78 and a diagonal one 0.65 of that per stage (TMA kernel; measured), plus
    // a fixed prologue/epilogue per CTA and a term per split for the second-stage reduction.  (Wave quantisation was
    // 14 % of the first nano profile at S = 2.)
    const int sms = prop.multiProcessorCount;
    const bool tma_likely = !(cfg->flags & RT_NO_TMA) && (Ng % 2 == 0) && get_encode_fn() != nullptr;
    const bool narrow = tma_likely && ntile > 1 && (N - (ntile - 1) * TILE) <= 96;
    p.Tn = narrow ? ntile - 1 : 0;
    p.Tfull = ntile * (ntile - 1) / 2 - p.Tn;
    const double cost_n = 0.78, cost_d = tma_likely ? 0.65 : 1.0;
    // one stage ~ 2.1 us on one SM; the reduction reads one N x ldn slab per split at ~3 TB/s
    const double cta_ovh = 8.0, split_ovh = (double)N * ldn * 8.0 / 3.0e12 / 2.1e-6;
    const long long kmin = 16 * 8;
    long long smax = (Ng + kmin - 1) / kmin;
    if (smax > 4 * sms) smax = 4 * sms;
    const double slab_bytes = (double)N * ldn * 8;
    // workspace cap: 2 GB, or up to 6 GB when the device has room after everything else (24k: S = 3 slabs of 1.35 GB
    // turn the half-empty 36th wave of 5,253 one-shot tiles into balanced waves, ~1 % of a 5.5 s kernel)
    double ws_cap = 2.0e9;
    {
      size_t freeb = 0, totalb = 0;
      if (cudaMemGetInfo(&freeb, &totalb) == cudaSuccess) {
        const double other = 16.0 * (double)c->nn_alloc * 8 + ((double)ntile + 1) / 2 * Ng * 8 + 14.0 * NgF * 8 +
                             ((cfg->flags & RT_PHI_DEVICE) ? 0.0 : (double)N * Ng * 8);
        const double room = 0.5 * ((double)freeb - other);
        if (room > ws_cap) ws_cap = room < 6.0e9 ? room : 6.0e9;
      } else {
        cudaGetLastError();
      }
    }
    while (smax > 1 && smax * slab_bytes > ws_cap) --smax;
    auto chunk_of = [&](long long S_) { long long kc = (Ng + S_ - 1) / S_; return (kc + 15) / 16 * 16; };
    auto makespan = [&](const long long (&n)[3], const double (&cst)[3]) {
      std::priority_queue<double, std::vector<double>, std::greater<double>> q;
      for (int i = 0; i < sms; ++i) q.push(0.0);
      double end = 0.0;
      for (int cls = 0; cls < 3; ++cls)
        for (long long j = 0; j < n[cls]; ++j) {
          const double t = q.top() + cst[cls];
          q.pop();
          q.push(t);
          if (t > end) end = t;
        }
      return end;
    };
    double best = 1e300;
    p.S = p.Sn = p.Sd = 1;
    p.kchunk = p.kchunk_n = p.kchunk_d = chunk_of(1);
    for (long long s = 1; s <= smax; ++s) {
      const long long kc = chunk_of(s);
      const long long S_ = (Ng + kc - 1) / kc;
      if (S_ != s) continue;                                       // same chunk as a smaller s
      const long long sn0 = p.Tn ? (long long)std::llround(cost_n * (double)s) : 1;
      const long long sd0 = (long long)std::llround(cost_d * (double)s);
      for (long long sn = sn0 - 1; sn <= sn0 + 1; ++sn) {
        if (sn < 1 || sn > s || (!p.Tn && sn != sn0)) continue;
        const long long kn = chunk_of(sn);
        const long long Sn_ = (Ng + kn - 1) / kn;
        for (long long sd = sd0 - 1; sd <= sd0 + 1; ++sd) {
          if (sd < 1 || sd > s) continue;
          const long long kd = chunk_of(sd);
          const long long Sd_ = (Ng + kd - 1) / kd;
          const long long cnt[3] = {S_ * p.Tfull, Sn_ * p.Tn, Sd_ * ntile};
          const double cst[3] = {kc / 16.0 + cta_ovh, cost_n * kn / 16.0 + cta_ovh, cost_d * kd / 16.0 + cta_ovh};
          const long long smost = p.Tfull > 0 ? S_ : (p.Tn > 0 ? Sn_ : Sd_);
          const double obj = makespan(cnt, cst) + split_ovh * (double)smost;
          if (obj < best - 1e-9) {
            best = obj;
            p.S = (int)S_; p.kchunk = kc; p.Sn = (int)Sn_; p.kchunk_n = kn; p.Sd = (int)Sd_; p.kchunk_d = kd;
          }
        }
      }
    }
    DensityPlan& d = c->dp;
    d.N = N; d.Ng = Ng; d.ntile = ntile; d.npairs = (ntile + 1) / 2; d.nrt = (Ng + TILE - 1) / TILE; d.ldn = ldn;
    // work types of the TMA kernel: one per pair.  (Cutting the pairs' time lines into several types per r-tile, so
    // that fewer Phi panels are in flight, was measured on nano: 4 pieces -> 397 ms and 277 GB of DRAM reads against
    // 364 ms and 191 GB for whole pairs; the extra epilogues and pipeline refills cost more than the locality buys.)
    const int nsplit = 1;
    c->dens_resident = 0.5 * (double)N * ldn * 8 <= 24.0e6;          // the fold stays in L2: raster regime (a) below
    build_density_types(N, ntile, nsplit, !c->dens_resident, c->segs);
    d.ntypes = (int)(c->segs.size() / 2);
    // Raster (gemm_tma.cu dens_decode), two regimes, both measured with ncu (profiles/r2_traffic.md):
    // (a) the fold stays in L2 (<= 24 MB, N <= ~2,400): ALL types of a small group of r-tiles run side by side and the Phi
    //     column panels of the r-tiles in flight are kept resident with the evict_last hint on their TMA loads -- every
    //     type re-reads its own k-range of a panel at its own time, and re-reading the fold costs nothing.
    //     nano: 72 GB of DRAM reads per launch (Phi = 40 GB) against 238 GB for the round-1 raster.
    // (b) larger N: the fold streams, the L2 cannot hold panels of N rows for the ~2 ms an item lives (measured: hints or
    //     not, 7.1-7.6 TB per launch at N = 13,000 = every item fetching its own panel).  Supertiles of group_t types x
    //     group_r r-tiles (~ one item per SM) then run in LOCK-STEP (producer pacing, gemm_tma.cu): a fold tile is fetched
    //     once for the group_r CTAs of its type and -- thanks to the type-independent k order of build_density_types -- a
    //     Phi tile once for the group_t CTAs of its r-tile, in each of the two passes (down, up) over k:
    //         DRAM bytes ~ 2 |Phi| ceil(ntypes / group_t) + |P fold| ceil(nrt / group_r)
    //     24k: 1.25 TB per launch against 7.2 TB, L2 hit rate 78 % against 34 %, kernel time +0.5 %.
    {
      const double phi_b = (double)N * Ng * 8, pf_b = 0.5 * (double)N * ldn * 8, panel = (double)N * TILE * 8;
      if (c->dens_resident) {
        long long gr = (long long)(10.0e6 / panel);
        d.group_t = d.ntypes;
        d.group_r = (int)std::max(1LL, std::min((long long)d.nrt, gr));
      } else {
        double best_cost = 1e300;
        d.group_t = 1; d.group_r = 1;
        for (int gt = 1; gt <= d.ntypes && gt <= sms; ++gt) {
          long long gr = sms / gt;
          if (gr > d.nrt) gr = d.nrt;
          if (gr < 1) gr = 1;
          const double cost = 2.0 * phi_b * std::ceil((double)d.ntypes / gt) + pf_b * std::ceil((double)d.nrt / (double)gr);
          if (cost < best_cost - 1.0) { best_cost = cost; d.group_t = gt; d.group_r = (int)gr; }
        }
      }
    }
  }

  // memory check, then allocations
  {
    size_t freeb = 0, totalb = 0;
    CKC(cudaMemGetInfo(&freeb, &totalb));
    double need = 15.0 * (double)c->nn_alloc * 8 + (double)c->pp.S * N * ldn * 8 + (double)c->dp.ntypes * Ng * 8 + 12.0 * NgF * 8;
    if (!(cfg->flags & RT_PHI_DEVICE)) need += (double)N * Ng * 8;
    if (need > (double)freeb) {
      char buf[256];
      snprintf(buf, sizeof buf, "rt_create: needs %.2f GB of device memory, %.2f GB free", need / 1e9, freeb / 1e9);
      FAIL_CREATE(RT_ENOMEM, buf);
    }
  }
  if (cfg->flags & RT_PHI_DEVICE) {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, phi) != cudaSuccess || pa.type != cudaMemoryTypeDevice) {
      cudaGetLastError();
      FAIL_CREATE(RT_EINVAL, "rt_create: RT_PHI_DEVICE set but phi is not a device pointer");
    }
    c->phi = phi;
  } else {
    ALLOC(c->phi_owned, (size_t)N * Ng);
    CKC(cudaMemcpyAsync(c->phi_owned, phi, (size_t)N * Ng * 8, cudaMemcpyHostToDevice, c->st));
    c->phi = c->phi_owned;
  }
  c->sms = prop.multiProcessorCount;
  c->use_tma = !(cfg->flags & RT_NO_TMA) && (Ng % 2 == 0) && ((reinterpret_cast<uintptr_t>(c->phi) & 15) == 0) &&
               get_encode_fn() != nullptr;
  if (c->use_tma) {
    if (!make_map(&c->tmPhiK, c->phi, N, Ng, Ng, BK_HOST, TILE)) c->use_tma = false;
    else if (make_map_phi3d(&c->tmPhiN, c->phi, N, Ng)) c->phiN_3d = 1;
    else if (!make_map(&c->tmPhiN, c->phi, N, Ng, Ng, 16, BK_HOST)) c->use_tma = false;
  }
  if (c->use_h) {
    if ((int)c->lv.size() > MG_MAX_LEVELS) FAIL_CREATE(RT_EINVAL, "rt_create: too many multigrid levels");
    const int e = init_mg_kernels();
    if (e != 0) FAIL_CREATE(RT_ECUDA, std::string("init_mg_kernels: ") + cudaGetErrorString((cudaError_t)e));
  }
  if (c->use_tma) {
    const int e = init_tma_kernels();
    if (e != 0) FAIL_CREATE(RT_ECUDA, std::string("init_tma_kernels: ") + cudaGetErrorString((cudaError_t)e));
  }
  const size_t nn = c->nn_alloc;        // N x ldn, rows padded so that every rank's row block has the same size
  ALLOC(c->d_eps, N); ALLOC(c->d_occ, N); ALLOC(c->d_E, 8); ALLOC(c->d_energy, 8);
  c->hist_cap = cfg->history;
  if (c->hist_cap) {
    ALLOC(c->d_hist, (size_t)c->hist_cap * 4);
    CKC(cudaMemsetAsync(c->d_hist, 0, (size_t)c->hist_cap * 32, c->st));
    ALLOC(c->d_hist_n, 1);
    CKC(cudaMemsetAsync(c->d_hist_n, 0, sizeof(unsigned long long), c->st));
  }
  ALLOC(c->d_bsums, 5 * 1024);
  if (c->prop == RT_PROP_COMMUTATOR || c->dynamic) {
    ALLOC(c->d_cs, 1);
    CKC(cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st));
  }
  double** mats[] = {&c->Hm1, &c->H0, &c->H1, &c->X, &c->Ya, &c->Yb, &c->Yc, &c->Cm, &c->Sc, &c->Sm,
                     &c->P0r, &c->P0i, &c->P1r, &c->P1i};
  for (double** mp : mats) { ALLOC(*mp, nn); CKC(cudaMemsetAsync(*mp, 0, nn * 8, c->st)); }
  ALLOC(c->W, (size_t)c->pp.S * N * ldn);
  if (c->prop == RT_PROP_TAYLOR && !c->general && c->q >= 4 && c->q <= SERIES_MAX_Q) {
    // the higher powers of Y, when they fit next to everything else with 2 GB to spare (else the products accumulate)
    size_t fb = 0, tb = 0;
    if (cudaMemGetInfo(&fb, &tb) == cudaSuccess && (double)fb > (double)(c->q - 3) * nn * 8 + 2.0e9) {
      for (int k = 4; k <= c->q; ++k) {
        double* pwk = nullptr;
        ALLOC(pwk, nn);
        CKC(cudaMemsetAsync(pwk, 0, nn * 8, c->st));
        c->pw_extra.push_back(pwk);
      }
    } else {
      cudaGetLastError();
    }
  }
  if (Hks_in) { ALLOC(c->Hks, nn); CKC(cudaMemsetAsync(c->Hks, 0, nn * 8, c->st)); }
  if (c->general) {
    double** extra[] = {&c->Rt, &c->It, c->magnus >= 2 ? &c->Wm : nullptr, c->nonorth ? &c->Smat : nullptr,
                        c->nonorth ? &c->Sinv : nullptr, c->nonorth ? &c->Bm : nullptr};
    for (double** mp : extra)
      if (mp) { ALLOC(*mp, nn); CKC(cudaMemsetAsync(*mp, 0, nn * 8, c->st)); }
  }
  // rho and the five sums share one allocation: it is the first exchange buffer of the slab mode
  ALLOC(c->rho, NgF + 8); ALLOC(c->rho0, NgF); ALLOC(c->vxc0, NgF);
  c->d_sums = c->rho + NgF;
  CKC(cudaMemsetAsync(c->rho, 0, (size_t)(NgF + 8) * 8, c->st));
  ALLOC(c->w, NgF + 16); ALLOC(c->op_u, NgF + 16);    // projection weights: the TMA path reads whole 16-double stages
  CKC(cudaMemsetAsync(c->w, 0, (size_t)(NgF + 16) * 8, c->st));
  CKC(cudaMemsetAsync(c->op_u, 0, (size_t)(NgF + 16) * 8, c->st));
  ALLOC(c->rho_part, (size_t)c->dp.ntypes * Ng);
  if (c->xc_kind == RT_XC_PBE) {
    ALLOC(c->pbe_scr, 4 * (size_t)NgF); ALLOC(c->vxc_cur, NgF); ALLOC(c->exc_a, NgF); ALLOC(c->exc_b, NgF);
  }
  if (c->fd_order == 4 && c->use_h) {
    ALLOC(c->f4, NgF);
    c->dl0 = c->lv[0];
    ALLOC(c->dl0.u, NgF); ALLOC(c->dl0.tmp, NgF); ALLOC(c->dl0.f, NgF); ALLOC(c->dl0.r, NgF);
    CKC(cudaMemsetAsync(c->dl0.u, 0, (size_t)NgF * 8, c->st));
  }
  ALLOC(c->d_segs, c->segs.size());
  CKC(cudaMemcpyAsync(c->d_segs, c->segs.data(), c->segs.size() * sizeof(DensSeg), cudaMemcpyHostToDevice, c->st));
  for (size_t l = 0; l < c->lv.size(); ++l) {
    MgLevel& L = c->lv[l];
    ALLOC(L.u, L.n); ALLOC(L.tmp, L.n); ALLOC(L.f, L.n); ALLOC(L.r, L.n);
    CKC(cudaMemsetAsync(L.u, 0, (size_t)L.n * 8, c->st));
  }
  {
    std::vector<int2> tiles;
    // full off-diagonal tiles, then the narrow last column (if any), then the diagonal (ProjectPlan)
    // The full tiles in 2-D blocks of bs x bs tiles (bs^2 ~ number of SMs): the CTAs of a wave then share bs row panels and
    // bs column panels of Phi in L2 instead of streaming one private
    // column panel each -- at N = 13,000 a row-major list made every one of the 5,151 tiles read its own 1.15 GB panel.
    const int tj_end = c->pp.Tn > 0 ? ntile - 1 : ntile;
    int bs = (int)std::floor(std::sqrt((double)c->sms));
    if (bs < 1) bs = 1;
    for (int bi = 0; bi < ntile; bi += bs)
      for (int bj = bi; bj < tj_end; bj += bs)
        for (int ti = bi; ti < std::min(bi + bs, ntile); ++ti)
          for (int tj = std::max(bj, ti + 1); tj < std::min(bj + bs, tj_end); ++tj) tiles.push_back(make_int2(ti, tj));
    if (c->pp.Tn > 0)
      for (int ti = 0; ti < ntile - 1; ++ti) tiles.push_back(make_int2(ti, ntile - 1));
    for (int ti = 0; ti < ntile; ++ti) tiles.push_back(make_int2(ti, ti));
    ALLOC(c->d_tiles, tiles.size());
    CKC(cudaMemcpyAsync(c->d_tiles, tiles.data(), tiles.size() * sizeof(int2), cudaMemcpyHostToDevice, c->st));
    std::vector<int2> full;
    for (int ti = 0; ti < ntile; ++ti)
      for (int tj = 0; tj < ntile; ++tj) full.push_back(make_int2(ti, tj));
    ALLOC(c->d_tiles_full, full.size());
    CKC(cudaMemcpyAsync(c->d_tiles_full, full.data(), full.size() * sizeof(int2), cudaMemcpyHostToDevice, c->st));
    std::vector<int2> symrm;
    for (int ti = 0; ti < ntile; ++ti)
      for (int tj = ti; tj < ntile; ++tj) symrm.push_back(make_int2(ti, tj));
    ALLOC(c->d_tiles_sym, symrm.size());
    CKC(cudaMemcpyAsync(c->d_tiles_sym, symrm.data(), symrm.size() * sizeof(int2), cudaMemcpyHostToDevice, c->st));
    if (c->use_tma) {
      // checkpoint counters of the paced launches (one array serves both kernels: they never run together on a handle)
      const size_t np = std::max(project_tma_pace_ints(c->pp, c->sms),
                                 c->dens_resident ? (size_t)0 : density_tma_pace_ints(c->dp, c->sms));
      if (np > 0) ALLOC(c->pace_cnt, np);
    }
    if (c->use_tma && N > GEMM_SMALL_N) {
      ALLOC(c->gemm_ws, gemm_tma_ws_doubles(c->sms));
      ALLOC(c->gemm_sync, gemm_tma_sync_ints(c->sms));
      CKC(cudaMemsetAsync(c->gemm_sync, 0, gemm_tma_sync_ints(c->sms) * sizeof(int), c->st));
    }
    CKC(cudaStreamSynchronize(c->st));
  }
  {
    const MgLevel& L = c->lv.back();
    std::vector<double> Q, lam;
    double** qs[3] = {&c->Qx, &c->Qy, &c->Qz};
    double** ls[3] = {&c->lx, &c->ly, &c->lz};
    const int dims[3] = {L.gd.nx, L.gd.ny, L.gd.nz};
    for (int d = 0; d < 3; ++d) {
      eigenbasis_1d(dims[d], L.h, Q, lam);
      ALLOC(*qs[d], Q.size()); ALLOC(*ls[d], lam.size());
      CKC(cudaMemcpy(*qs[d], Q.data(), Q.size() * 8, cudaMemcpyHostToDevice));
      CKC(cudaMemcpy(*ls[d], lam.data(), lam.size() * 8, cudaMemcpyHostToDevice));
    }
  }
  CKC(cudaMemcpy(c->d_eps, eps, (size_t)N * 8, cudaMemcpyHostToDevice));
  if (occ) CKC(cudaMemcpy(c->d_occ, occ, (size_t)N * 8, cudaMemcpyHostToDevice));
  else CKC(cudaMemset(c->d_occ, 0, (size_t)N * 8));
  {
    double e8[8] = {cfg->E0[0], cfg->E0[1], cfg->E0[2], 0, 0, 0, 0, 0};
    CKC(cudaMemcpy(c->d_E, e8, sizeof e8, cudaMemcpyHostToDevice));
  }

  // non-orthogonal basis: overlap S = dVol Phi Phi^T (Eq. 30) by the projection kernel with unit weights, then S^-1
  // by the Newton-Schulz iteration X <- X (2 - S X) on the N x N GEMM kernels (every iterate is a polynomial in S:
  // symmetric outputs), started from X0 = S / (|S|_1 |S|_inf), stopped when max|S X - 1| <= 1e-14
  if (c->nonorth) {
    std::vector<double> ones((size_t)NgF + 16, 1.0);
    CKC(cudaMemcpyAsync(c->w, ones.data(), ((size_t)NgF + 16) * 8, cudaMemcpyHostToDevice, c->st));
    enqueue_project(c, c->w, nullptr, c->Smat);
    std::vector<double> Sh((size_t)N * ldn);
    CKC(cudaMemcpyAsync(Sh.data(), c->Smat, Sh.size() * 8, cudaMemcpyDeviceToHost, c->st));
    CKC(cudaStreamSynchronize(c->st));
    double n1 = 0.0;
    for (int i = 0; i < N; ++i) {
      double r = 0.0;
      for (int j = 0; j < N; ++j) r += std::fabs(Sh[(size_t)i * ldn + j]);
      n1 = std::fmax(n1, r);
    }
    if (!(n1 > 0.0) || !std::isfinite(n1)) FAIL_CREATE(RT_EINVAL, "rt_create: the overlap matrix dVol Phi Phi^T is zero or non-finite");
    launch_axpby(N, ldn, 1.0 / (n1 * n1), c->Smat, 0.0, c->Smat, c->Sinv, c->st);       // X0 (S symmetric: |S|_1 = |S|_inf)
    // X <- 2 X - (X S) X.  The iterate is mirrored from its upper triangle after every update: with X exactly symmetric the
    // error obeys E <- -E S E; without it the antisymmetric rounding noise doubles every iteration and the iteration blows
    // up a few steps after it has converged (measured).  Stop at 1e-13, or when the residual stagnates at its rounding floor.
    double res = 1.0, prev = 2.0;
    int itn = 0;
    for (; itn < 100; ++itn) {
      enqueue_gemm(c, 0, c->Sinv, c->Smat, 1.0, nullptr, nullptr, 0, c->Rt);            // T = X S
      CKC(cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st));
      launch_maxabs_minus_identity(N, ldn, c->Rt, c->d_cs, c->st);
      ConvState hs;
      CKC(cudaMemcpyAsync(&hs, c->d_cs, sizeof hs, cudaMemcpyDeviceToHost, c->st));
      CKC(cudaStreamSynchronize(c->st));
      memcpy(&res, &hs.H_bits, 8);
      if (!std::isfinite(res) || res <= 1e-13 || (res < 1e-8 && res > 0.5 * prev)) break;
      prev = res;
      enqueue_gemm(c, 0, c->Rt, c->Sinv, 1.0, nullptr, nullptr, 0, c->It);              // (X S) X
      launch_axpby(N, ldn, 2.0, c->Sinv, -1.0, c->It, c->Sinv, c->st);
      launch_hermitize(N, ldn, c->Sinv, c->It, c->st);                                  // mirror X (It is scratch)
    }
    c->newton_iters = itn;
    if (!(res <= 1e-10)) {
      char buf[200];
      snprintf(buf, sizeof buf, "rt_create: the overlap matrix could not be inverted (Phi linearly dependent?): "
               "max|S X - 1| = %.3e after %d Newton-Schulz iterations, |S|_1 = %.3e", res, itn, n1);
      FAIL_CREATE(RT_EINVAL, buf);
    }
    CKC(cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st));
  }

  // initial state (Alg. 1 lines 7-8): P0 = diag(occ); rho0; vxc0; H0 = H-1 = diag(eps) + Proj(E0.r)
  if (P0re_in) {
    if (int rc = copy_matrix_in(c, P0re_in, c->P0r)) { std::string m_ = c->err; FAIL_CREATE(rc, m_); }
    if (P0im_in) { if (int rc = copy_matrix_in(c, P0im_in, c->P0i)) { std::string m_ = c->err; FAIL_CREATE(rc, m_); } }
  } else {
    launch_set_diag(N, ldn, c->P0r, c->d_occ, c->st);
  }
  if (Hks_in) { if (int rc = copy_matrix_in(c, Hks_in, c->Hks)) { std::string m_ = c->err; FAIL_CREATE(rc, m_); } }
  launch_field(NgF, c->gd, c->h, c->d_E, c->w, c->st);
  if (!c->slab) {
    enqueue_density(c, c->P0r, c->rho0, nullptr);
    CKC(cudaMemcpyAsync(c->rho, c->rho0, (size_t)Ng * 8, cudaMemcpyDeviceToDevice, c->st));
    enqueue_vxc(c, c->rho0, c->vxc0);
    enqueue_project(c, c->w, c->d_eps, c->H0);
    CKC(cudaMemcpyAsync(c->Hm1, c->H0, nn * 8, cudaMemcpyDeviceToDevice, c->st));
    CKC(cudaMemcpyAsync(c->H1, c->H0, nn * 8, cudaMemcpyDeviceToDevice, c->st));
    // sums[4] currently holds sum(rho0) (rho0 pointer was NULL): the induced charge at t = 0 is zero
    CKC(cudaMemsetAsync(c->d_sums + 4, 0, 8, c->st));
    enqueue_record(c);                                             // time level 0
  } else {
    // slab: the local pieces go to the exchange buffers; RT_SLAB_INIT finishes after the caller's all-reduce
    enqueue_density(c, c->P0r, c->rho + c->slab_off, nullptr);
    enqueue_project_dv(c, c->H1);
  }
  {
    double z8[8] = {0, 0, 0, 0, 0, 0, 0, 0};                  // E(t_1) defaults to 0 (DESIGN R5)
    CKC(cudaMemcpyAsync(c->d_E, z8, sizeof z8, cudaMemcpyHostToDevice, c->st));
  }
  CKC(cudaStreamSynchronize(c->st));
  CKC(cudaGetLastError());

  // capture one step into a CUDA graph (pointers are fixed: line 28 is a copy, not a pointer rotation).  With
  // H_thrs > 0 the number of updates is decided on the host, so the unit captured is one Hamiltonian update.
  {
    const int64_t before = c->launches;
    if (c->use_graph && !c->slab) {
      // capture on a private stream (the caller's may be the legacy default stream, which cannot capture);
      // the instantiated graph is replayed on the caller's stream
      // A capture can be invalidated from outside the library (another host thread of the process; seen with several
      // handles driven by host threads on one GPU): it is retried, and after three failures the handle simply launches
      // its kernels directly -- the graph is an optimisation, not a requirement.
      cudaStream_t user = c->st, cap = nullptr;
      CKC(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
      c->st = cap;
      cudaError_t e = cudaSuccess;
      for (int attempt = 0; attempt < 3; ++attempt) {
        e = cudaSuccess;
        c->launches = before;
        if (!c->dynamic) {
          e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
          if (e == cudaSuccess) {
            enqueue_step(c);
            e = cudaStreamEndCapture(cap, &c->graph);
          }
          c->launches_per_step = c->launches - before;
        } else {
          for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            const int64_t b0 = c->launches;
            e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
              enqueue_update(c, i);
              e = cudaStreamEndCapture(cap, &c->graph_upd[i]);
            }
            c->launches_per_upd[i] = c->launches - b0;
          }
        }
        if (e == cudaSuccess) break;
        cudaGetLastError();
        c->capture_failures += 1;
        if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
        for (int i = 0; i < 2; ++i)
          if (c->graph_upd[i]) { cudaGraphDestroy(c->graph_upd[i]); c->graph_upd[i] = nullptr; }
      }
      c->st = user;
      cudaStreamDestroy(cap);
      if (e == cudaSuccess) {
        if (c->graph) CKC(cudaGraphInstantiate(&c->gexec, c->graph, 0));
        for (int i = 0; i < 2; ++i)
          if (c->graph_upd[i]) CKC(cudaGraphInstantiate(&c->gexec_upd[i], c->graph_upd[i], 0));
      }
    }
    c->launches = before;
  }
#undef ALLOC
#undef CKC
#undef FAIL_CREATE
  *out = c;
  return RT_OK;
}
}  // namespace

extern "C" {

int rt_create(const rt_config* cfg, const double* phi, const double* eps, const double* occ, rt_handle* out) {
  if (!occ) return fail(nullptr, RT_EINVAL, "rt_create: NULL argument");
  return create_impl(cfg, phi, eps, occ, nullptr, nullptr, nullptr, out);
}

int rt_create_general(const rt_config* cfg, const double* phi, const double* eps, const double* Hks, const double* P0re,
                      const double* P0im, rt_handle* out) {
  if (!Hks || !P0re) return fail(nullptr, RT_EINVAL, "rt_create_general: NULL argument");
  return create_impl(cfg, phi, eps, nullptr, Hks, P0re, P0im, out);
}

int rt_set_field(rt_handle c, const double E[3]) {
  CHECK_HANDLE(c);
  if (!E) return fail(c, RT_EINVAL, "rt_set_field: NULL");
  const double e0 = E[0], e1 = E[1], e2 = E[2];                 // read now: the value travels as a kernel argument
  if (!(e0 == e0 && e1 == e1 && e2 == e2)) return fail(c, RT_EINVAL, "rt_set_field: NaN");
  // The Taylor degree q / the commutator kmax were fixed at rt_create from the spectral bound with E0 (DESIGN R8):
  // refuse a field that takes the truncation term of that fixed order above 1e-15 (design bound 1e-17).
  {
    const double theta = c->theta0 + c->dt * (std::fabs(e0) * c->half_len[0] + std::fabs(e1) * c->half_len[1] +
                                               std::fabs(e2) * c->half_len[2]);
    bool ok = true;
    if (c->prop == RT_PROP_TAYLOR && c->cfg.exp_order == 0) {
      double term = 1.0;
      for (int k = 1; k <= 2 * c->q + 2; ++k) term *= theta / k;
      ok = term <= 1e-15;
    } else if (c->prop == RT_PROP_COMMUTATOR && c->cfg.max_order == 0) {
      double term = 2.0;
      for (int k = 1; k <= c->kmax; ++k) term *= 2.0 * theta / k;
      ok = term <= c->dP_thrs;
    }
    if (!ok) return fail(c, RT_EINVAL, "rt_set_field: |E| exceeds the bound the series order was sized for at rt_create "
                                       "(create the handle with E0 of that magnitude or with an explicit exp_order / max_order)");
  }
  CK(cudaSetDevice(c->cfg.device));
  launch_set_field(c->d_E, e0, e1, e2, c->st);
  c->launches += 1;
  CK(cudaGetLastError());
  return RT_OK;
}

int rt_step(rt_handle c, int32_t nsteps) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_step: slab handle -- drive it with rt_slab_phase");
  if (nsteps < 0) return fail(c, RT_EINVAL, "rt_step: nsteps < 0");
  CK(cudaSetDevice(c->cfg.device));
  for (int s = 0; s < nsteps; ++s) {
    if (c->dynamic) {
      // Alg. 1 lines 12-26: while (H_err > H_thrs).  The decision needs H_err on the host: one 8-byte read and a
      // stream synchronisation per Hamiltonian update.
      int it = 0;
      double herr = 2.0 * c->H_thrs;
      while (herr > c->H_thrs && it < c->max_hup) {
        const int kind = it == 0 ? 0 : 1;
        if (c->gexec_upd[kind] && !c->timing) {
          CK(cudaGraphLaunch(c->gexec_upd[kind], c->st));
          c->launches += c->launches_per_upd[kind];
        } else {
          enqueue_update(c, kind);
          CK(cudaGetLastError());
        }
        ConvState hs;
        CK(cudaMemcpyAsync(&hs, c->d_cs, sizeof hs, cudaMemcpyDeviceToHost, c->st));
        if (int rc = sync_and_check(c)) return rc;
        memcpy(&herr, &hs.H_bits, 8);
        c->last_orders = hs.k_used;
        memcpy(&c->last_dP_err, &hs.dP_bits[hs.k_used], 8);
        ++it;
        if (!std::isfinite(herr) || !std::isfinite(c->last_dP_err)) {
          c->last_hupdates = it; c->last_H_err = herr;
          return fail(c, RT_ENUMERIC, "rt_step: non-finite H1 or dP (time step too large for the series, or bad input)");
        }
        if (c->prop == RT_PROP_COMMUTATOR && !hs.done) {
          c->last_hupdates = it; c->last_H_err = herr;
          return fail(c, RT_ENUMERIC, "rt_step: the commutator series did not reach dP_thrs within max_order terms");
        }
      }
      enqueue_shift(c);
      CK(cudaGetLastError());
      c->last_hupdates = it;
      c->last_H_err = herr;
    } else if (c->gexec && !c->timing) {
      CK(cudaGraphLaunch(c->gexec, c->st));
      c->launches += c->launches_per_step;
    } else {
      const int64_t before = c->launches;
      enqueue_step(c);
      if (!c->launches_per_step) c->launches_per_step = c->launches - before;
      CK(cudaGetLastError());
    }
    c->t += c->dt;
    c->steps_done += 1;
  }
  return RT_OK;
}

int rt_get_dipole_series(rt_handle c, int64_t first, int32_t n, double* out) {
  CHECK_HANDLE(c);
  if (!out || n < 0 || first < 0) return fail(c, RT_EINVAL, "rt_get_dipole_series: bad argument");
  if (!c->hist_cap) return fail(c, RT_EINVAL, "rt_get_dipole_series: handle created with history = 0");
  const int64_t have = c->steps_done + 1;                  // levels 0 .. steps_done
  if (first + n > have || first < have - c->hist_cap || first < c->hist_first)
    return fail(c, RT_EINVAL, "rt_get_dipole_series: requested levels are not in the history window");
  CK(cudaSetDevice(c->cfg.device));
  for (int32_t i = 0; i < n;) {                            // at most two contiguous pieces of the ring
    const int64_t slot = (first + i) % c->hist_cap;
    int32_t run = (int32_t)((c->hist_cap - slot < n - i) ? (c->hist_cap - slot) : (n - i));
    CK(cudaMemcpyAsync(out + (size_t)i * 4, c->d_hist + slot * 4, (size_t)run * 32, cudaMemcpyDeviceToHost, c->st));
    i += run;
  }
  return sync_and_check(c);
}

int rt_get_convergence(rt_handle c, int32_t n[2], double err[2]) {
  CHECK_HANDLE(c);
  if (!n || !err) return fail(c, RT_EINVAL, "rt_get_convergence: NULL");
  CK(cudaSetDevice(c->cfg.device));
  n[0] = c->dynamic ? c->last_hupdates : c->m;
  n[1] = 0;
  err[0] = c->dynamic ? c->last_H_err : 0.0;
  err[1] = 0.0;
  if (c->d_cs && c->prop == RT_PROP_COMMUTATOR) {
    if (c->dynamic) { n[1] = c->last_orders; err[1] = c->last_dP_err; }
    else {
      ConvState hs;
      CK(cudaMemcpyAsync(&hs, c->d_cs, sizeof hs, cudaMemcpyDeviceToHost, c->st));
      if (int rc = sync_and_check(c)) return rc;
      n[1] = hs.k_used;
      memcpy(&err[1], &hs.dP_bits[hs.k_used], 8);
      if (c->steps_done > 0 && (!std::isfinite(err[1]) || !hs.done))
        return fail(c, RT_ENUMERIC, "rt_get_convergence: the last commutator series is non-finite or stopped at max_order above dP_thrs");
    }
  }
  return RT_OK;
}

int rt_get_dipole(rt_handle c, double mu[3]) {
  CHECK_HANDLE(c);
  if (!mu) return fail(c, RT_EINVAL, "rt_get_dipole: NULL");
  CK(cudaSetDevice(c->cfg.device));
  double s[5];
  CK(cudaMemcpyAsync(s, c->d_sums, sizeof s, cudaMemcpyDeviceToHost, c->st));
  if (int rc = sync_and_check(c)) return rc;
  for (int q = 0; q < 3; ++q) mu[q] = c->dvol * s[1 + q];
  return RT_OK;
}

int rt_get_charge(rt_handle c, double q[2]) {
  CHECK_HANDLE(c);
  if (!q) return fail(c, RT_EINVAL, "rt_get_charge: NULL");
  CK(cudaSetDevice(c->cfg.device));
  double s[5];
  CK(cudaMemcpyAsync(s, c->d_sums, sizeof s, cudaMemcpyDeviceToHost, c->st));
  if (int rc = sync_and_check(c)) return rc;
  q[0] = c->dvol * s[0];
  q[1] = c->dvol * s[4];
  return RT_OK;
}

int rt_get_density(rt_handle c, double* rho) {
  CHECK_HANDLE(c);
  if (!rho) return fail(c, RT_EINVAL, "rt_get_density: NULL");
  CK(cudaSetDevice(c->cfg.device));
  CK(cudaMemcpyAsync(rho, c->rho, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  return sync_and_check(c);
}

// ---- checkpoint / resume ---------------------------------------------------------------------------
namespace {
struct StateHeader { uint64_t magic; int32_t norb, nx, ny, nz; double dt, t; int64_t steps; int64_t ndoubles; };
static_assert(sizeof(StateHeader) <= 64, "header must fit its 64-byte slot");
constexpr uint64_t STATE_MAGIC = 0x3130455441545352ull;          // "RSTATE01"
int64_t state_doubles(const rt_ctx* c) { return 4LL * c->N * c->N + 2LL * c->Ng + 16; }
}  // namespace

int rt_state_bytes(rt_handle c, int64_t* nbytes) {
  CHECK_HANDLE(c);
  if (!nbytes) return fail(c, RT_EINVAL, "rt_state_bytes: NULL");
  *nbytes = 64 + 8 * state_doubles(c);
  return RT_OK;
}

int rt_get_state(rt_handle c, void* buf) {
  CHECK_HANDLE(c);
  if (!buf) return fail(c, RT_EINVAL, "rt_get_state: NULL");
  if (c->slab && c->slab_state != 1) return fail(c, RT_ESTATE, "rt_get_state: RT_SLAB_INIT has not run");
  CK(cudaSetDevice(c->cfg.device));
  StateHeader hd{STATE_MAGIC, c->N, c->gd.nx, c->gd.ny, c->gd.nz, c->dt, c->t, c->steps_done, state_doubles(c)};
  memset(buf, 0, 64);
  memcpy(buf, &hd, sizeof hd);
  double* p = reinterpret_cast<double*>(static_cast<char*>(buf) + 64);
  const size_t n2 = (size_t)c->N * c->N;
  const double* mats[4] = {c->P0r, c->P0i, c->H0, c->Hm1};
  for (int i = 0; i < 4; ++i)
    if (int rc = copy_matrix_out(c, mats[i], p + i * n2)) return rc;
  p += 4 * n2;
  CK(cudaMemcpyAsync(p, c->lv[0].u, (size_t)c->Ng * 8, cudaMemcpyDeviceToHost, c->st));
  CK(cudaMemcpyAsync(p + c->Ng, c->rho, (size_t)c->Ng * 8, cudaMemcpyDeviceToHost, c->st));
  CK(cudaMemcpyAsync(p + 2 * c->Ng, c->d_sums, 8 * 8, cudaMemcpyDeviceToHost, c->st));
  CK(cudaMemcpyAsync(p + 2 * c->Ng + 8, c->d_E, 8 * 8, cudaMemcpyDeviceToHost, c->st));
  return sync_and_check(c);
}

int rt_set_state(rt_handle c, const void* buf) {
  CHECK_HANDLE(c);
  if (!buf) return fail(c, RT_EINVAL, "rt_set_state: NULL");
  if (c->slab && c->slab_state != 1) return fail(c, RT_ESTATE, "rt_set_state: RT_SLAB_INIT has not run");
  StateHeader hd;
  memcpy(&hd, buf, sizeof hd);
  if (hd.magic != STATE_MAGIC || hd.norb != c->N || hd.nx != c->gd.nx || hd.ny != c->gd.ny || hd.nz != c->gd.nz ||
      hd.dt != c->dt || hd.ndoubles != state_doubles(c))
    return fail(c, RT_EINVAL, "rt_set_state: the buffer was not written by a handle with this norb / grid / dt");
  CK(cudaSetDevice(c->cfg.device));
  const double* p = reinterpret_cast<const double*>(static_cast<const char*>(buf) + 64);
  const size_t n2 = (size_t)c->N * c->N;
  double* mats[4] = {c->P0r, c->P0i, c->H0, c->Hm1};
  for (int i = 0; i < 4; ++i)
    if (int rc = copy_matrix_in(c, p + i * n2, mats[i])) return rc;
  p += 4 * n2;
  CK(cudaMemcpyAsync(c->lv[0].u, p, (size_t)c->Ng * 8, cudaMemcpyHostToDevice, c->st));
  CK(cudaMemcpyAsync(c->rho, p + c->Ng, (size_t)c->Ng * 8, cudaMemcpyHostToDevice, c->st));
  CK(cudaMemcpyAsync(c->d_sums, p + 2 * c->Ng, 8 * 8, cudaMemcpyHostToDevice, c->st));
  CK(cudaMemcpyAsync(c->d_E, p + 2 * c->Ng + 8, 8 * 8, cudaMemcpyHostToDevice, c->st));
  // H1 is rebuilt from H0 and H-1 by the first update of the next step (line 11); P1 by the propagation
  c->t = hd.t;
  c->steps_done = hd.steps;
  c->hist_first = hd.steps;
  if (c->hist_cap) {                                   // the history restarts at this level
    const unsigned long long k = (unsigned long long)hd.steps;
    CK(cudaMemcpyAsync(c->d_hist_n, &k, sizeof k, cudaMemcpyHostToDevice, c->st));
    if (int rc = sync_and_check(c)) return rc;
    enqueue_record(c);
  }
  return sync_and_check(c);
}

int rt_get_energy(rt_handle c, double* energy) {
  CHECK_HANDLE(c);
  if (!energy) return fail(c, RT_EINVAL, "rt_get_energy: NULL");
  if (c->slab && c->slab_state != 1) return fail(c, RT_ESTATE, "rt_get_energy: RT_SLAB_INIT has not run");
  CK(cudaSetDevice(c->cfg.device));
  if (c->xc_kind == RT_XC_PBE && c->use_xc) {
    launch_vxc_pbe(c->gd, c->h, c->fd_order, c->rho, c->pbe_scr, nullptr, c->exc_a, c->st);     // e_xc(rho), e_xc(rho0)
    launch_vxc_pbe(c->gd, c->h, c->fd_order, c->rho0, c->pbe_scr, nullptr, c->exc_b, c->st);
    launch_energy_exc(c->Ng, c->gd, c->h, c->rho, c->rho0, c->vxc0, c->lv[0].u, c->d_E, c->exc_a, c->exc_b, c->use_h, c->N,
                      c->ldn, c->d_eps, c->P0r, c->d_bsums, c->d_energy, c->st);
    c->launches += 2;
  } else {
    launch_energy(c->Ng, c->gd, c->h, c->rho, c->rho0, c->vxc0, c->lv[0].u, c->d_E, c->use_h, c->use_xc, c->N, c->ldn,
                  c->d_eps, c->P0r, c->d_bsums, c->d_energy, c->st);
  }
  c->launches += 3;
  if (c->Hks) {                                      // tr(H_KS Re P) replaces sum_i eps_i Re P_ii
    launch_trace_product(c->N, c->ldn, c->Hks, c->P0r, c->d_energy, c->st);
    c->launches += 1;
  }
  double out[8];
  CK(cudaMemcpyAsync(out, c->d_energy, sizeof out, cudaMemcpyDeviceToHost, c->st));
  if (int rc = sync_and_check(c)) return rc;
  *energy = out[5] + c->dvol * out[0];
  return RT_OK;
}

int rt_get_vhartree(rt_handle c, double* vh) {
  CHECK_HANDLE(c);
  if (!vh) return fail(c, RT_EINVAL, "rt_get_vhartree: NULL");
  CK(cudaSetDevice(c->cfg.device));
  CK(cudaMemcpyAsync(vh, c->lv[0].u, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  return sync_and_check(c);
}

int rt_get_pmatrix(rt_handle c, double* re, double* im) {
  CHECK_HANDLE(c);
  CK(cudaSetDevice(c->cfg.device));
  if (int rc = copy_matrix_out(c, c->P0r, re)) return rc;
  if (int rc = copy_matrix_out(c, c->P0i, im)) return rc;
  return sync_and_check(c);
}

int rt_get_hmatrix(rt_handle c, double* H0) {
  CHECK_HANDLE(c);
  CK(cudaSetDevice(c->cfg.device));
  if (int rc = copy_matrix_out(c, c->H0, H0)) return rc;
  return sync_and_check(c);
}

int rt_get_overlap(rt_handle c, double* S, double* Sinv) {
  CHECK_HANDLE(c);
  if (!c->nonorth) return fail(c, RT_EINVAL, "rt_get_overlap: handle was created without RT_NONORTHOGONAL");
  CK(cudaSetDevice(c->cfg.device));
  if (int rc = copy_matrix_out(c, c->Smat, S)) return rc;
  if (int rc = copy_matrix_out(c, c->Sinv, Sinv)) return rc;
  return sync_and_check(c);
}

int rt_get_time(rt_handle c, double* t) {
  CHECK_HANDLE(c);
  if (!t) return fail(c, RT_EINVAL, "rt_get_time: NULL");
  *t = c->t;
  return RT_OK;
}

int rt_get_info(rt_handle c, int32_t info[8]) {
  CHECK_HANDLE(c);
  if (!info) return fail(c, RT_EINVAL, "rt_get_info: NULL");
  const MgLevel& L = c->lv.back();
  info[0] = 2 * c->q + 1;
  info[1] = (int32_t)c->lv.size();
  info[2] = L.gd.nx; info[3] = L.gd.ny; info[4] = L.gd.nz;
  info[5] = ((c->gexec || !c->phase_exec.empty()) ? 1 : 0) | (c->use_tma ? 2 : 0) | (c->capture_failures > 0 ? 4 : 0) |
            ((c->use_tma && c->pace_cnt && project_tma_pace_ints(c->pp, c->sms) > 0) ? 8 : 0) |
            ((c->use_tma && c->pace_cnt && !c->dens_resident && density_tma_pace_ints(c->dp, c->sms) > 0) ? 16 : 0);
  info[6] = (int32_t)c->launches_per_step;
  info[7] = c->pp.S;
  return RT_OK;
}

int rt_get_launch_count(rt_handle c, int64_t* n) {
  CHECK_HANDLE(c);
  if (!n) return fail(c, RT_EINVAL, "rt_get_launch_count: NULL");
  *n = c->launches;
  return RT_OK;
}

// ---- per-stage entry points ------------------------------------------------------------------------
int rt_op_project(rt_handle c, const double* v, double* out) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_op_project: not available on a slab handle");
  if (!v || !out) return fail(c, RT_EINVAL, "rt_op_project: NULL");
  CK(cudaSetDevice(c->cfg.device));
  CK(cudaMemcpyAsync(c->op_u, v, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  stage_begin(c, RT_STAGE_HUPDATE);
  enqueue_project(c, c->op_u, nullptr, c->Ya);
  stage_end(c);
  if (int rc = copy_matrix_out(c, c->Ya, out)) return rc;
  return sync_and_check(c);
}

int rt_op_density(rt_handle c, const double* reP, double* rho, double sums[5]) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_op_density: not available on a slab handle");
  if (!reP || !rho) return fail(c, RT_EINVAL, "rt_op_density: NULL");
  CK(cudaSetDevice(c->cfg.device));
  if (int rc = copy_matrix_in(c, reP, c->Ya)) return rc;
  // d_sums is propagation state (dipole of the current density): save and restore around the call
  double keep[5];
  CK(cudaMemcpyAsync(keep, c->d_sums, sizeof keep, cudaMemcpyDeviceToHost, c->st));
  stage_begin(c, RT_STAGE_RHO);
  enqueue_density(c, c->Ya, c->op_u, c->rho0);
  stage_end(c);
  double s[5];
  CK(cudaMemcpyAsync(s, c->d_sums, sizeof s, cudaMemcpyDeviceToHost, c->st));
  CK(cudaMemcpyAsync(rho, c->op_u, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  if (int rc = sync_and_check(c)) return rc;
  CK(cudaMemcpyAsync(c->d_sums, keep, sizeof keep, cudaMemcpyHostToDevice, c->st));
  if (int rc = sync_and_check(c)) return rc;
  if (sums) memcpy(sums, s, sizeof s);
  return RT_OK;
}

int rt_op_propagate(rt_handle c, const double* Hbar, const double* P0re, const double* P0im, double* P1re,
                    double* P1im) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_op_propagate: not available on a slab handle");
  if (!Hbar || !P0re || !P0im || !P1re || !P1im) return fail(c, RT_EINVAL, "rt_op_propagate: NULL");
  if (c->general) return fail(c, RT_EINVAL, "rt_op_propagate: takes one Hbar; not defined for magnus_order = 2 / RT_NONORTHOGONAL");
  CK(cudaSetDevice(c->cfg.device));
  const size_t nn = (size_t)c->N * c->ldn;
  // The propagation state owns Hm1/H0/H1/P0/P1 and the series owns X..Sm: the call needs five more N x N matrices.
  // They are allocated once per handle, on first use, and freed by rt_destroy.
  if (!c->op_T[0]) {
    double* T5 = nullptr;
    if (int rc = dev_alloc(c, &T5, 5 * nn)) return rc;
    for (int i = 0; i < 5; ++i) c->op_T[i] = T5 + i * nn;
  }
  double** T = c->op_T;
  if (int rc = copy_matrix_in(c, Hbar, T[0])) return rc;
  if (int rc = copy_matrix_in(c, P0re, T[1])) return rc;
  if (int rc = copy_matrix_in(c, P0im, T[2])) return rc;
  stage_begin(c, RT_STAGE_ELDYN);
  launch_hbar(c->N, c->ldn, T[0], T[0], T[0], c->X, c->dt, c->sigma, 0, c->st);   // X = dt (Hbar - sigma I)
  c->launches += 1;
  if (c->d_cs) cudaMemsetAsync(c->d_cs, 0, sizeof(ConvState), c->st);
  enqueue_propagate(c, T[1], T[2], T[3], T[4]);
  stage_end(c);
  if (int rc = copy_matrix_out(c, T[3], P1re)) return rc;
  if (int rc = copy_matrix_out(c, T[4], P1im)) return rc;
  return sync_and_check(c);
}

int rt_op_hartree(rt_handle c, double* vh, const double* drho, int32_t n_vc) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_op_hartree: not available on a slab handle");
  if (!vh || !drho || n_vc < 0) return fail(c, RT_EINVAL, "rt_op_hartree: bad argument");
  if (!c->use_h) return fail(c, RT_EINVAL, "rt_op_hartree: handle created with RT_NO_HARTREE");
  CK(cudaSetDevice(c->cfg.device));
  double keep[5];
  CK(cudaMemcpyAsync(keep, c->d_sums, sizeof keep, cudaMemcpyDeviceToHost, c->st));
  // run the cycle on a private level-0 solution (op_u) and rhs input staged in w
  CK(cudaMemcpyAsync(c->op_u, vh, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  CK(cudaMemcpyAsync(c->w, drho, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  std::vector<MgLevel> lv = c->lv;
  lv[0].u = c->op_u;
  stage_begin(c, RT_STAGE_VH);
  launch_sum_only(c->w, c->Ng, c->d_bsums, c->d_sums, c->st);
  c->launches += 2;
  enqueue_poisson(c, lv, n_vc, c->w, nullptr);
  stage_end(c);
  CK(cudaMemcpyAsync(vh, c->op_u, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  if (int rc = sync_and_check(c)) return rc;
  CK(cudaMemcpyAsync(c->d_sums, keep, sizeof keep, cudaMemcpyHostToDevice, c->st));
  return sync_and_check(c);
}

int rt_op_vxc(rt_handle c, const double* rho, double* vxc) {
  CHECK_HANDLE(c);
  if (c->slab) return fail(c, RT_ESTATE, "rt_op_vxc: not available on a slab handle");
  if (!rho || !vxc) return fail(c, RT_EINVAL, "rt_op_vxc: NULL");
  CK(cudaSetDevice(c->cfg.device));
  CK(cudaMemcpyAsync(c->op_u, rho, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  stage_begin(c, RT_STAGE_XC);
  enqueue_vxc(c, c->op_u, c->w);
  stage_end(c);
  CK(cudaMemcpyAsync(vxc, c->w, (size_t)c->Ng * 8, cudaMemcpyDefault, c->st));
  return sync_and_check(c);
}

// ---- grid-slab sharding -----------------------------------------------------------------------------
int rt_slab_get_buffers(rt_handle c, rt_slab_buffers* out) {
  CHECK_HANDLE(c);
  if (!out) return fail(c, RT_EINVAL, "rt_slab_get_buffers: NULL");
  if (!c->slab) return fail(c, RT_ESTATE, "rt_slab_get_buffers: handle was created without a slab");
  out->xchg_rho = c->rho;
  out->xchg_rho_count = c->Ng + 8;
  out->xchg_H = c->H1;
  out->xchg_H_count = (int64_t)c->N * c->ldn;
  out->slab_offset = c->slab_off;
  out->slab_count = c->Ngl;
  return RT_OK;
}

int rt_slab_get_shard(rt_handle c, rt_shard_buffers* out) {
  CHECK_HANDLE(c);
  if (!out) return fail(c, RT_EINVAL, "rt_slab_get_shard: NULL");
  if (!c->slab) return fail(c, RT_ESTATE, "rt_slab_get_shard: handle was created without a slab");
  out->Y = c->Ya; out->C = c->Cm; out->S = c->Sm; out->P1re = c->P1r; out->P1im = c->P1i;
  out->block_count = (int64_t)c->shard_rows * c->ldn;
  out->total_count = (int64_t)c->nn_alloc;
  out->prop_shards = c->nshard;
  out->prop_shard = c->shard;
  return RT_OK;
}

int rt_slab_more_updates(rt_handle c, int32_t* more) {
  CHECK_HANDLE(c);
  if (!more) return fail(c, RT_EINVAL, "rt_slab_more_updates: NULL");
  if (!c->slab) return fail(c, RT_ESTATE, "rt_slab_more_updates: handle was created without a slab");
  *more = c->slab_more;
  return RT_OK;
}

namespace {
// one phase of the slab protocol, enqueued on c->st (directly, or while that stream is capturing)
void enqueue_slab_phase(rt_ctx* c, int phase, int it) {
  switch (phase) {
    case RT_SLAB_PROPAGATE: enqueue_update_propagate(c, it); break;
    case RT_SLAB_PROP_A: enqueue_shard_A(c, it); break;
    case RT_SLAB_PROP_B: enqueue_shard_B(c); break;
    case RT_SLAB_PROP_C: enqueue_shard_C(c); break;
    case RT_SLAB_PROP_D:
      launch_hermitize(c->N, c->ldn, c->P1r, c->P1i, c->st);
      c->launches += 1;
      enqueue_density_stage(c);
      break;
    case RT_SLAB_POTENTIAL: enqueue_update_potential(c); break;
    case RT_SLAB_SHIFT: enqueue_shift(c); break;
    default: break;
  }
}
}  // namespace

int rt_slab_phase(rt_handle c, int32_t phase, int32_t it) {
  CHECK_HANDLE(c);
  if (!c->slab) return fail(c, RT_ESTATE, "rt_slab_phase: handle was created without a slab");
  CK(cudaSetDevice(c->cfg.device));
  const size_t nn = (size_t)c->N * c->ldn * 8;
  if (phase != RT_SLAB_INIT && c->slab_state != 1) return fail(c, RT_ESTATE, "rt_slab_phase: RT_SLAB_INIT has not run");
  if (it < 0) return fail(c, RT_EINVAL, "rt_slab_phase: it < 0");
  switch (phase) {
    case RT_SLAB_INIT:            // xchg_rho holds rho0 of the whole grid, xchg_H holds H(t = 0)  (Alg. 1 lines 7-8)
      if (c->slab_state != 0) return fail(c, RT_ESTATE, "rt_slab_phase: RT_SLAB_INIT already done");
      CK(cudaMemcpyAsync(c->rho0, c->rho, (size_t)c->Ng * 8, cudaMemcpyDeviceToDevice, c->st));
      enqueue_vxc(c, c->rho0, c->vxc0);
      CK(cudaMemcpyAsync(c->H0, c->H1, nn, cudaMemcpyDeviceToDevice, c->st));
      CK(cudaMemcpyAsync(c->Hm1, c->H1, nn, cudaMemcpyDeviceToDevice, c->st));
      CK(cudaMemsetAsync(c->d_sums + 4, 0, 8, c->st));       // induced charge at t = 0
      enqueue_record(c);                                     // time level 0
      c->slab_state = 1;
      break;
    case RT_SLAB_PROPAGATE:
      if (c->nshard > 1) return fail(c, RT_ESTATE, "rt_slab_phase: a handle with prop_shards > 1 propagates with RT_SLAB_PROP_A..D");
      goto enqueue;
    case RT_SLAB_PROP_A: case RT_SLAB_PROP_B: case RT_SLAB_PROP_C: case RT_SLAB_PROP_D:
      if (c->nshard <= 1) return fail(c, RT_ESTATE, "rt_slab_phase: RT_SLAB_PROP_A..D need prop_shards > 1");
      goto enqueue;
    case RT_SLAB_POTENTIAL:
    case RT_SLAB_SHIFT:
    enqueue: {
      // The phases are fixed launch sequences: each (phase, first-update?) pair is captured once into a CUDA graph on a
      // private stream and replayed afterwards (one launch instead of ~50 at the small configs).
      const bool last = c->dynamic || it >= c->m - 1;          // the last update also forms Im P1 (enqueue_upu)
      const int key = 4 * phase + 2 * (it == 0 ? 1 : 0) + (last ? 1 : 0);
      if (c->use_graph && !c->timing) {
        auto ex = c->phase_exec.find(key);
        // A capture can be invalidated from outside the library (another host thread of the process synchronising the
        // device or using the legacy stream in a way the capture mode forbids).  The graph is only an optimisation: a
        // failed capture is discarded, the phase is enqueued directly this time, and the capture is tried again on the
        // next use (three times per phase at most).
        if (ex == c->phase_exec.end() && c->phase_capture_failures[key] < 3) {
          cudaStream_t user = c->st, cap = nullptr;
          CK(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
          c->st = cap;
          const int64_t before = c->launches;
          cudaGraph_t g = nullptr;
          cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
          if (e == cudaSuccess) {
            enqueue_slab_phase(c, phase, it);
            e = cudaStreamEndCapture(cap, &g);
          }
          c->phase_launches[key] = c->launches - before;
          c->launches = before;
          c->st = user;
          cudaStreamDestroy(cap);
          cudaGraphExec_t gx = nullptr;
          if (e == cudaSuccess) e = cudaGraphInstantiate(&gx, g, 0);
          if (e != cudaSuccess) {
            cudaGetLastError();
            if (g) cudaGraphDestroy(g);
            c->phase_capture_failures[key] += 1;
            c->capture_failures += 1;
          } else {
            c->phase_graphs.push_back(g);
            ex = c->phase_exec.emplace(key, gx).first;
          }
        }
        if (ex != c->phase_exec.end()) {
          CK(cudaGraphLaunch(ex->second, c->st));
          c->launches += c->phase_launches[key];
        } else {
          enqueue_slab_phase(c, phase, it);
        }
      } else {
        enqueue_slab_phase(c, phase, it);
      }
      if (phase == RT_SLAB_SHIFT) { c->t += c->dt; c->steps_done += 1; }
      if (phase == RT_SLAB_POTENTIAL && !c->dynamic) { c->slab_more = (it + 1 < c->m) ? 1 : 0; c->last_hupdates = it + 1; }
      break;
    }
    case RT_SLAB_CHECK: {
      // Alg. 1 lines 12-13 / 24 on a sharded system: xchg_H now holds the complete H1 (after the caller's all-reduce)
      // and Ya the previous one; the norm is a max over replicated, bit-identical matrices, so every rank takes the
      // same decision without another collective.  Fixed-count handles just count.
      if (!c->dynamic) { c->slab_more = (it + 1 < c->m) ? 1 : 0; break; }
      launch_maxabs_diff(c->N, c->ldn, c->H1, c->Ya, c->d_cs, c->st);
      c->launches += 1;
      ConvState hs;
      CK(cudaMemcpyAsync(&hs, c->d_cs, sizeof hs, cudaMemcpyDeviceToHost, c->st));
      if (int rc = sync_and_check(c)) return rc;
      double herr;
      memcpy(&herr, &hs.H_bits, 8);
      c->last_H_err = herr;
      c->last_hupdates = it + 1;
      if (!std::isfinite(herr)) return fail(c, RT_ENUMERIC, "rt_slab_phase: non-finite H1");
      c->slab_more = (herr > c->H_thrs && it + 1 < c->max_hup) ? 1 : 0;
      break;
    }
    default:
      return fail(c, RT_EINVAL, "rt_slab_phase: unknown phase");
  }
  CK(cudaGetLastError());
  return RT_OK;
}

int rt_spectrum(const double* mu, int32_t nt, double dt, double t_kick, const double kappa[3], double gamma,
                const double* omega, int32_t nw, double* S, int32_t device, void* stream) {
  rt_ctx* c = nullptr;
  if (!mu || !kappa || !omega || !S || nt < 2 || nw < 0 || !(dt > 0.0) || !(gamma >= 0.0))
    return fail(c, RT_EINVAL, "rt_spectrum: bad argument");
  int nused = 0;
  for (int q = 0; q < 3; ++q) nused += kappa[q] != 0.0;
  if (!nused) return fail(c, RT_EINVAL, "rt_spectrum: every kappa is zero");
  if (nw == 0) return RT_OK;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  cudaError_t e = cudaSetDevice(device);
  double *d_mu = nullptr, *d_w = nullptr, *d_S = nullptr;
  auto is_dev = [](const void* p) {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return pa.type == cudaMemoryTypeDevice || pa.type == cudaMemoryTypeManaged;
  };
  const bool mu_dev = is_dev(mu), w_dev = is_dev(omega), S_dev = is_dev(S);
  if (e == cudaSuccess && !mu_dev) { e = cudaMalloc(&d_mu, (size_t)3 * nt * 8); if (e == cudaSuccess) e = cudaMemcpyAsync(d_mu, mu, (size_t)3 * nt * 8, cudaMemcpyHostToDevice, st); }
  if (e == cudaSuccess && !w_dev) { e = cudaMalloc(&d_w, (size_t)nw * 8); if (e == cudaSuccess) e = cudaMemcpyAsync(d_w, omega, (size_t)nw * 8, cudaMemcpyHostToDevice, st); }
  if (e == cudaSuccess && !S_dev) e = cudaMalloc(&d_S, (size_t)nw * 8);
  if (e == cudaSuccess) {
    launch_spectrum(mu_dev ? mu : d_mu, nt, dt, t_kick, kappa, nused, gamma, w_dev ? omega : d_w, nw, S_dev ? S : d_S, st);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess && !S_dev) e = cudaMemcpyAsync(S, d_S, (size_t)nw * 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_mu); cudaFree(d_w); cudaFree(d_S);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(c, RT_ECUDA, std::string("rt_spectrum: ") + cudaGetErrorString(e)); }
  return RT_OK;
}

int rt_spectrum_kick(const double* mu, int32_t nt, double dt, const double E_kick[3], double gamma, const double* omega,
                     int32_t nw, double* S, int32_t device, void* stream) {
  if (!E_kick) return fail(nullptr, RT_EINVAL, "rt_spectrum_kick: NULL");
  // end-point sampled kick (DESIGN R5): the trapezoid of Alg. 1 line 14 delivers E dt / 2 at the effective time dt / 2
  const double kappa[3] = {0.5 * E_kick[0] * dt, 0.5 * E_kick[1] * dt, 0.5 * E_kick[2] * dt};
  return rt_spectrum(mu, nt, dt, 0.5 * dt, kappa, gamma, omega, nw, S, device, stream);
}

int rt_dipole_noalloc(const double* rho, int32_t nx, int32_t ny, int32_t nz, double h, double* out, int32_t device,
                      void* stream) {
  if (!rho || !out || nx < 1 || ny < 1 || nz < 1 || !(h > 0.0))
    return fail(nullptr, RT_EINVAL, "rt_dipole_noalloc: bad argument");
  static_assert(RT_NOALLOC_MAX_POINTS == 4096LL * 1024LL, "header limit and noalloc.cu disagree");
  if (dipole_noalloc_max_points() != RT_NOALLOC_MAX_POINTS)
    return fail(nullptr, RT_EINVAL, "rt_dipole_noalloc: header limit and library limit disagree");
  std::string err;
  const int rc = launch_dipole_noalloc(rho, nx, ny, nz, h, out, device, reinterpret_cast<cudaStream_t>(stream), &err);
  if (rc != RT_OK) return fail(nullptr, rc, err);
  return RT_OK;
}

int rt_timing_enable(rt_handle c, int32_t enable) {
  CHECK_HANDLE(c);
  c->timing = enable != 0;
  return RT_OK;
}

int rt_timing_read(rt_handle c, double ms[RT_STAGE_COUNT], int64_t calls[RT_STAGE_COUNT]) {
  CHECK_HANDLE(c);
  CK(cudaSetDevice(c->cfg.device));
  if (int rc = sync_and_check(c)) return rc;
  if (int rc = collect_timing(c)) return rc;
  for (int i = 0; i < RT_STAGE_COUNT; ++i) {
    if (ms) ms[i] = c->stage_ms[i];
    if (calls) calls[i] = c->stage_calls[i];
    c->stage_ms[i] = 0;
    c->stage_calls[i] = 0;
  }
  return RT_OK;
}

}  // extern "C"
