// api.cu -- the C ABI of librism3d.so (include/rism3d.h): context, workspace carving, argument checks, and
// the launch sequence of one iteration.  No arithmetic of the method lives here except
// the host-side preparation of small input tables (twiddles, mixed LJ parameters).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "rism3d_internal.h"

using namespace r3d;

struct rism3d_ctx {
  rism3d_params p;
  Grid g;
  Buffers b;
  SolverParams sp;
  cudaStream_t stream;
  char* ws;
  size_t ws_bytes;
  size_t scratch_bytes;      // bytes of the X..work span that set_* may use for uploads
  bool have_solvent, have_solute;
  double qv[MAX_NV], sigv[MAX_NV], epsv[MAX_NV], rhov[MAX_NV], gramw[MAX_NV];
  long long launches;
  bool profiling;            // per-kernel CUDA-event timing of the loop kernels (rism3d_set_profiling)
  std::vector<cudaEvent_t>* ev_pool;
  size_t ev_used;
  double prof_ms[RISM3D_N_LOOP_KERNELS];
  long long prof_iters;
  // CUDA graphs of 1 and of GRAPH_PACK iterations (captured once per context: every launch parameter of an
  // iteration is fixed, all evolving state lives on the device); not used on the legacy default stream or while profiling
  cudaGraphExec_t graph1, graph_pack;
  bool graph_tried;
  int graph_kernels;         // kernels per captured iteration
  std::vector<double>* h_atoms;   // host copies of the solute tables (x, y, z, .) and (beta C q q, sigma^2, 4 beta eps)
  std::vector<double>* h_pair;    //   kept for rism3d_gradient: their device copies live in scratch the loop overwrites
  int n_atoms;
  bool phi_valid;            // phi(r) has been computed for the current solute (with a cutoff it is computed when first
                             // needed: the loop never reads it)
  float phi_ms;              // GPU time of that deferred phi kernel
  StateHeader* h_hdr;        // pinned
  double* d_out;             // small device array for scalar results (inside workspace)
  bool peer_broken;          // an in-stream barrier of a peer-mode iterate timed out: reconnect before iterating again
  char err[512];
};

static int fail(rism3d_ctx* c, int code, const char* fmt, ...) {
  if (c) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c->err, sizeof(c->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

#define CU(call)                                                                                        \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess) return fail(ctx, RISM3D_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

// Every entry point that touches the GPU runs on the context's device, whatever device is current in the calling
// thread, and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  bool ok = true;            // false: `dev` could not be made current -- the caller must not go on (it would work on
                             // whatever device happens to be current)
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev) {
      switched = (cudaSetDevice(dev) == cudaSuccess);
      ok = switched;
    }
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define ON_CTX_DEVICE(ctx)                        \
  DeviceGuard device_guard_((ctx)->p.device);     \
  if (!device_guard_.ok) return fail(ctx, RISM3D_ERR_CUDA, "device %d could not be made current", (ctx)->p.device)

// small RAII holders so that an early return through CU() does not leak
struct ScopedEvents {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaError_t create() {
    cudaError_t e = cudaEventCreate(&e0);
    return e != cudaSuccess ? e : cudaEventCreate(&e1);
  }
  ~ScopedEvents() {
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
  }
};
struct ScopedDeviceAlloc {
  void* p = nullptr;
  ~ScopedDeviceAlloc() {
    if (p) cudaFree(p);
  }
};

static bool device_exists(int device) {
  int n = 0;
  return cudaGetDeviceCount(&n) == cudaSuccess && device >= 0 && device < n;
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// TMA descriptor of a row-major 2D array of doubles [rows][row_len] with row pitch `pitch_bytes`, boxes of
// box_rows x box_cols elements (cuTensorMapEncodeTiled, looked up through the runtime: no link-time libcuda)
static bool make_tensor_map_2d(CUtensorMap* tm, void* base, uint64_t row_len, uint64_t rows, uint64_t pitch_bytes,
                               uint32_t box_cols, uint32_t box_rows) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || fn == nullptr ||
      qres != cudaDriverEntryPointSuccess)
    return false;
  const cuuint64_t dims[2] = {row_len, rows};
  const cuuint64_t strides[1] = {pitch_bytes};
  const cuuint32_t box[2] = {box_cols, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  return ((encode_fn)fn)(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// kernels are instantiated for 1, 2, 4 and 8 site types (the sites of a k point share 8 / nv-wide tile rows and are
// exchanged by butterfly shuffles): other counts run padded with phantom types
static int padded_sites(int nv) { return nv <= 1 ? 1 : (nv <= 2 ? 2 : (nv <= 4 ? 4 : 8)); }

static bool pow2_in(int n, int lo, int hi) { return n >= lo && n <= hi && (n & (n - 1)) == 0; }

static bool valid_params(const rism3d_params* p) {
  if (!p) return false;
  // every axis a power of two in 8..512, one spacing: the three lengths may differ (a box is rarely a cube)
  if (!pow2_in(p->nx, 8, 512) || !pow2_in(p->ny, 8, 512) || !pow2_in(p->nz, 8, 512)) return false;
  if (p->n_sites < 1 || p->n_sites > MAX_NV) return false;
  const int nv = padded_sites(p->n_sites);
  if (((p->nz / 2) * nv) % 8) return false;         // tile rows are 8 complex wide
  if (p->mdiis_nvec < 1 || p->mdiis_nvec > MAX_M) return false;
  if (!(p->spacing > 0.0) || !(p->temperature > 0.0) || !(p->kappa > 0.0)) return false;
  // r_min = 0 (e.g. a zero-initialised struct) would put 1/0 into w for a grid point on an atom (Q11); the clamp must
  // also stay well inside the float range of the rsqrt seed.  The mixing parameter must be positive.
  if (!(p->r_min >= 1e-6) || !(p->r_min < 1e6) || !(p->mdiis_b > 0.0) || !(p->mdiis_b < 1e6)) return false;
  if (kspace_smem_bytes(p->nx, nv) <= 0 || kspace_smem_bytes(p->nx, nv) > 227 * 1024) return false;
  if (p->closure != RISM3D_KH && p->closure != RISM3D_PSE && p->closure != RISM3D_HNC) return false;
  if (p->closure == RISM3D_PSE && p->pse_order < 1) return false;
  if (p->accelerator != RISM3D_ACCEL_MDIIS && p->accelerator != RISM3D_ACCEL_ANDERSON) return false;
  if (p->mdiis_dynamic_b && !(p->mdiis_b_min > 0.0 && p->mdiis_b_max >= p->mdiis_b_min && p->mdiis_b_max < 1e6)) return false;
  if (p->n_ranks > 1) {                              // slab decomposition: whole bricks / tiles per rank
    const int P = p->n_ranks;
    if (P > MAX_RANKS || (P & (P - 1)) || p->rank < 0 || p->rank >= P) return false;
    if (p->nx % P || p->ny % P || (p->nx / P) % 8 || (p->ny / P) % 8) return false;
  } else if (p->n_ranks < 0 || (p->n_ranks <= 1 && p->rank != 0)) {
    return false;
  }
  return true;
}

// geometry of the context's grid from the caller's parameters (device attributes are filled in by rism3d_init)
static Grid make_grid(const rism3d_params* p) {
  Grid g{};
  g.nx = p->nx; g.ny = p->ny; g.nz = p->nz;
  g.nmax = g.nx > g.ny ? (g.nx > g.nz ? g.nx : g.nz) : (g.ny > g.nz ? g.ny : g.nz);
  const int ex = g.nmax / g.nx, ey = g.nmax / g.ny, ez = g.nmax / g.nz;
  g.wx = ex * ex; g.wy = ey * ey; g.wz = ez * ez;
  // largest shell index: every folded index at its maximum n_axis / 2 - 1
  auto top = [](int n, int w) { const long long hn = n / 2; return (long long)w * (hn - 1) * hn; };
  g.nshell = (int)((top(g.nx, g.wx) + top(g.ny, g.wy) + top(g.nz, g.wz)) / 2 + 1);
  g.nv = padded_sites(p->n_sites); g.nv_user = p->n_sites; g.h = p->spacing;
  for (int i = 0; i < 3; ++i) g.origin[i] = p->origin[i];
  g.n_ranks = p->n_ranks > 1 ? p->n_ranks : 1;
  g.rank = p->n_ranks > 1 ? p->rank : 0;
  g.nxl = g.nx / g.n_ranks; g.ix0 = g.rank * g.nxl;
  g.nyl = g.ny / g.n_ranks; g.jy0 = g.rank * g.nyl;
  g.npts = (size_t)g.nxl * g.ny * g.nz;
  g.npts_global = (size_t)g.nx * g.ny * g.nz;
  g.field = g.npts * g.nv;
  return g;
}

// stored (input, residual) pairs: mdiis_nvec, or 3 for the modified Anderson method (the newest + two histories)
static int effective_m(const rism3d_params* p) { return p->accelerator == RISM3D_ACCEL_ANDERSON ? 3 : p->mdiis_nvec; }

// carve the workspace; with base == nullptr only the total size is computed
static size_t carve(const rism3d_params* p, char* base, Buffers* b, double** d_out, size_t* scratch_bytes) {
  const Grid gq = make_grid(p);
  const size_t nv = (size_t)gq.nv, M = (size_t)effective_m(p);
  const size_t npts = gq.npts, field = gq.field;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* ptr = base ? base + off : nullptr; off += align256(bytes); return ptr; };
  char* st = take(sizeof(DevState));
  const size_t off_x = off;
  char* Z = take(M * field * 8);
  char* R = take(M * field * 8);
  char* tau = take(field * 8);
  char* w = take(field * 8);
  char* work = take(field * 8);
  const size_t scr = off - off_x;
  char* phi = take(npts * 8);
  char* phik = take(npts * 8);
  char* chis = take((size_t)gq.nshell * nv * nv * 8);
  char* tw = take(2 * (size_t)gq.nmax * 16);
  const size_t nblk = (size_t)zinv_ctas(gq);          // one Gram partial per zinv_residual CTA
  const size_t ngrp = (nblk + 63) / 64;
  char* gp = take(nblk * (MAX_M + 1) * 2 * 8);
  char* gp2 = take(ngrp * (MAX_M + 1) * 2 * 8);
  char* tk = take(ngrp * 4);
  char* fp = take((size_t)2 * FE_BLOCKS * MAX_NV * 2 * 8);
  char* qv = take(MAX_NV * 8);
  char* rv = take(MAX_NV * 8);
  char* gw = take(MAX_NV * 8);
  char* out = take(64 * 8);
  char *kb = work, *stg = nullptr, *gx = nullptr, *xf = nullptr;
  if (gq.n_ranks > 1) {                             // slab run: the k-space slab, the staging array, the exchange rows
    kb = take(field * 8);
    stg = take(field * 8);
    gx = take((size_t)MAX_RANKS * GRAM_SLOT * 2 * 8);
    xf = take((MAX_RANKS + 1) * sizeof(unsigned long long));
  }
  if (b) {
    b->kbuf = (double2*)kb; b->stage = (double2*)stg; b->gram_x = (double*)gx; b->xflags = (unsigned long long*)xf;
    b->state = (DevState*)st;
    b->Z = (double*)Z; b->R = (double*)R; b->tau = (double*)tau; b->w = (double*)w; b->work = (double2*)work;
    b->phi = (double*)phi; b->phik = (double2*)phik; b->chi_shell = (double*)chis; b->tw = (double2*)tw;
    b->gram_part = (double*)gp; b->gram_part2 = (double*)gp2; b->tickets = (unsigned*)tk; b->n_tickets = ngrp; b->fe_part = (double*)fp; b->qv = (double*)qv; b->rhov = (double*)rv; b->gram_w = (double*)gw;
    b->scratch = (double*)work;
  }
  if (d_out) *d_out = (double*)out;
  if (scratch_bytes) *scratch_bytes = scr;
  return off;
}

extern "C" size_t rism3d_workspace_bytes(const rism3d_params* p) {
  if (!valid_params(p)) return 0;
  return carve(p, nullptr, nullptr, nullptr, nullptr);
}

extern "C" const char* rism3d_status_string(int s) {
  switch (s) {
    case RISM3D_OK: return "ok";
    case RISM3D_ERR_ARG: return "bad argument";
    case RISM3D_ERR_SIZE: return "unsupported size";
    case RISM3D_ERR_ORDER: return "call out of order";
    case RISM3D_ERR_CHI_RANGE: return "chi table does not cover the grid's |k| range";
    case RISM3D_ERR_NEUTRAL: return "solvent not neutral";
    case RISM3D_ERR_WORKSPACE: return "workspace too small";
    case RISM3D_ERR_CUDA: return "CUDA error";
    case RISM3D_ERR_DIVERGED: return "iteration diverged";
    case RISM3D_ERR_PEER: return "a peer rank did not reach an in-stream barrier in time";
    default: return "unknown status";
  }
}

extern "C" const char* rism3d_last_error(const rism3d_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" long long rism3d_launch_count(const rism3d_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int rism3d_init(rism3d_ctx** out, const rism3d_params* p, void* d_workspace, size_t bytes, void* stream) {
  if (!out || !p || !d_workspace) return RISM3D_ERR_ARG;
  *out = nullptr;
  if (!valid_params(p)) return RISM3D_ERR_SIZE;
  const size_t need = carve(p, nullptr, nullptr, nullptr, nullptr);
  if (bytes < need) return RISM3D_ERR_WORKSPACE;
  if (((uintptr_t)d_workspace) & 255) return RISM3D_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= p->device || p->device < 0) return RISM3D_ERR_CUDA;
  DeviceGuard device_guard_(p->device);
  int cur_dev = -1, num_sms = 0, smem_optin = 0;
  if (cudaGetDevice(&cur_dev) != cudaSuccess || cur_dev != p->device) return RISM3D_ERR_CUDA;
  if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, p->device) != cudaSuccess || num_sms <= 0 ||
      cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, p->device) != cudaSuccess)
    return RISM3D_ERR_CUDA;
  if (kspace_smem_bytes(p->nx, padded_sites(p->n_sites)) > smem_optin) return RISM3D_ERR_SIZE;
  rism3d_ctx* ctx = new rism3d_ctx();
  memset(ctx, 0, sizeof(*ctx));
  ctx->p = *p;
  ctx->stream = (cudaStream_t)stream;
  ctx->ws = (char*)d_workspace;
  ctx->ws_bytes = bytes;
  carve(p, ctx->ws, &ctx->b, &ctx->d_out, &ctx->scratch_bytes);
  Grid& g = ctx->g;
  g = make_grid(p);
  g.num_sms = num_sms;
  g.smem_optin = smem_optin;
  SolverParams& sp = ctx->sp;
  sp.closure = p->closure;
  sp.pse_order = p->closure == RISM3D_PSE ? p->pse_order : 1;
  sp.M = effective_m(p); sp.b = p->mdiis_b; sp.restart = p->mdiis_restart;
  sp.accel = p->accelerator; sp.and_s1 = p->anderson_s[0]; sp.and_s2 = p->anderson_s[1];
  if (sp.accel == RISM3D_ACCEL_ANDERSON) sp.restart = 0.0;   // the paper's method has no restart rule
  sp.dyn_b = p->mdiis_dynamic_b != 0 && sp.accel == RISM3D_ACCEL_MDIIS;
  sp.b_min = p->mdiis_b_min; sp.b_max = p->mdiis_b_max;
  sp.kT = K_BOLTZMANN * p->temperature;
  sp.beta = 1.0 / sp.kT;
  sp.kappa = p->kappa; sp.r_min = p->r_min;
  // twiddle table exp(-i pi j / nmax), j < 2 nmax, from long double (an axis of length n reads every (nmax/n)-th entry)
  std::vector<double> tw(4 * (size_t)g.nmax);
  for (int j = 0; j < 2 * g.nmax; ++j) {
    const long double a = 3.14159265358979323846264338327950288L * (long double)j / (long double)g.nmax;
    tw[2 * j] = (double)cosl(a);
    tw[2 * j + 1] = (double)(-sinl(a));
  }
  if (kspace_uses_tma(g.nx)) {
    // k-space pass tiles: nx rows (jx) of 8 complex = 16 doubles of `work`, and the matching 8 / nv phi~ values per row
    const uint64_t row_w = (uint64_t)g.nyl * g.q() * 2, row_p = (uint64_t)g.nyl * (g.nz / 2) * 2;   // doubles per jx row
    const uint32_t box_rows = (uint32_t)(g.nx < 256 ? g.nx : 256);                         // TMA box limit; 512 = two boxes
    if (!make_tensor_map_2d(&ctx->b.tm_work, ctx->b.kbuf, row_w, (uint64_t)g.nx, row_w * 8, 16, box_rows) ||
        !make_tensor_map_2d(&ctx->b.tm_phik, ctx->b.phik, row_p, (uint64_t)g.nx, row_p * 8, (uint32_t)(2 * 8 / g.nv), box_rows)) {
      delete ctx;
      return RISM3D_ERR_CUDA;
    }
  }
  if (g.n_ranks > 1) {
    // staged exchange until rism3d_slab_set_peers: block d of the staging array takes the rows of rank d's slab on the
    // way in and holds the rows that came back from rank d on the way out; the Gram row goes into this rank's own array
    const size_t blk = (size_t)g.nxl * g.nyl * g.q();
    for (int r = 0; r < g.n_ranks; ++r) {
      ctx->b.fwd_dst[r] = ctx->b.stage + (size_t)r * blk;
      ctx->b.bwd_src[r] = ctx->b.stage + (size_t)r * blk;
    }
    ctx->b.gram_dst[0] = ctx->b.gram_x;
    ctx->b.n_gram_dst = 1;
    ctx->b.peer_mode = false;
    ctx->b.peer_timeout_ns = 30ull * 1000000000ull;        // rism3d_slab_set_peer_timeout
  }
  if (y_uses_tma(g.ny, g.n_ranks)) {
    const uint64_t row = (uint64_t)g.q() * 2;                                                // doubles per (ix, iy) row
    if (!make_tensor_map_2d(&ctx->b.tm_ywork, ctx->b.work, row, (uint64_t)g.nxl * g.ny, row * 8, 2 * (uint32_t)y_tile_cols(g), (uint32_t)g.ny)) {
      delete ctx;
      return RISM3D_ERR_CUDA;
    }
  }
  cudaError_t e = cudaMallocHost((void**)&ctx->h_hdr, sizeof(StateHeader));
  if (e == cudaSuccess && g.n_ranks > 1) e = cudaMemsetAsync(ctx->b.gram_x, 0, (size_t)MAX_RANKS * GRAM_SLOT * 16, ctx->stream);
  if (e == cudaSuccess && g.n_ranks > 1) e = cudaMemsetAsync(ctx->b.xflags, 0, (MAX_RANKS + 1) * sizeof(unsigned long long), ctx->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->b.tw, tw.data(), tw.size() * 8, cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctx->b.state, 0, sizeof(DevState), ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctx->b.tickets, 0, ctx->b.n_tickets * sizeof(unsigned), ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) {
    if (ctx->h_hdr) cudaFreeHost(ctx->h_hdr);
    delete ctx;
    return RISM3D_ERR_CUDA;
  }
  *out = ctx;
  return RISM3D_OK;
}

extern "C" void rism3d_destroy(rism3d_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard device_guard_(ctx->p.device);
  if (device_guard_.ok) cudaStreamSynchronize(ctx->stream);
  if (ctx->ev_pool) {
    for (cudaEvent_t e : *ctx->ev_pool) cudaEventDestroy(e);
    delete ctx->ev_pool;
  }
  delete ctx->h_atoms;
  delete ctx->h_pair;
  if (ctx->graph1) cudaGraphExecDestroy(ctx->graph1);
  if (ctx->graph_pack) cudaGraphExecDestroy(ctx->graph_pack);
  if (ctx->h_hdr) cudaFreeHost(ctx->h_hdr);
  delete ctx;
}

extern "C" int rism3d_set_solvent_chi(rism3d_ctx* ctx, const double* q, const double* sigma, const double* eps,
                                      const double* rho, int n_k, double dk, double k0, const double* chi) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!q || !sigma || !eps || !rho || !chi || n_k < 4 || !(dk > 0.0)) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  const Grid& g = ctx->g;
  const int nu = g.nv_user;
  double neutral = 0.0;
  for (int i = 0; i < nu; ++i) neutral += rho[i] * q[i];
  if (fabs(neutral) > 1e-12) return fail(ctx, RISM3D_ERR_NEUTRAL, "sum rho_g q_g = %.3e", neutral);
  const double dkg = 2.0 * M_PI / (g.nmax * g.h), quarter_w = 0.25 * (g.wx + g.wy + g.wz);
  const double kmin = dkg * sqrt(quarter_w), kmax = dkg * sqrt(2.0 * (g.nshell - 1) + quarter_w);
  if ((kmin - k0) / dk < 0.0 || (kmax - k0) / dk > (double)(n_k - 1))
    return fail(ctx, RISM3D_ERR_CHI_RANGE, "table covers [%.4f, %.4f], grid needs [%.4f, %.4f]", k0,
                k0 + (n_k - 1) * dk, kmin, kmax);
  const size_t tbytes = (size_t)n_k * g.nv * g.nv * 8;
  for (int i = 0; i < g.nv; ++i) {                   // phantom types (i >= nu): no charge, no LJ well, no density
    const bool real = i < nu;
    ctx->qv[i] = real ? q[i] : 0.0; ctx->sigv[i] = real ? sigma[i] : 1.0; ctx->epsv[i] = real ? eps[i] : 0.0;
    ctx->rhov[i] = real ? rho[i] : 0.0;
  }
  std::vector<double> padded;                        // chi with zero rows and columns for the phantom types
  const double* table = chi;
  if (g.nv != nu) {
    padded.assign((size_t)n_k * g.nv * g.nv, 0.0);
    for (int m = 0; m < n_k; ++m)
      for (int a = 0; a < nu; ++a)
        for (int c = 0; c < nu; ++c) padded[((size_t)m * g.nv + a) * g.nv + c] = chi[((size_t)m * nu + a) * nu + c];
    table = padded.data();
  }
  // the radial table is only needed until chi_shell is built: it goes through the history span (rebuilt by set_solute
  // anyway) or, on grids too small to hold it, through a temporary allocation of the library's own
  double* d_table = ctx->b.Z;
  ScopedDeviceAlloc tmp;                             // freed on every way out, also an early CU() return
  if (tbytes > ctx->scratch_bytes) {
    CU(cudaMalloc(&tmp.p, tbytes));
    d_table = (double*)tmp.p;
  }
  CU(cudaMemcpyAsync(d_table, table, tbytes, cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaMemcpyAsync(ctx->b.qv, ctx->qv, g.nv * 8, cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaMemcpyAsync(ctx->b.rhov, ctx->rhov, g.nv * 8, cudaMemcpyHostToDevice, ctx->stream));
  for (int i = 0; i < g.nv; ++i)                   // inner-product weights: 1/rho_g for the modified Anderson method (Eq. 38)
    ctx->gramw[i] = (ctx->sp.accel == RISM3D_ACCEL_ANDERSON) ? (i < nu ? 1.0 / rho[i] : 0.0) : 1.0;
  CU(cudaMemcpyAsync(ctx->b.gram_w, ctx->gramw, g.nv * 8, cudaMemcpyHostToDevice, ctx->stream));
  ctx->launches += launch_chi_shell(g, ctx->b, d_table, n_k, k0, dk, ctx->stream);
  const cudaError_t e_launch = cudaGetLastError(), e_sync = cudaStreamSynchronize(ctx->stream);   // before tmp goes away
  CU(e_launch);
  CU(e_sync);
  ctx->have_solvent = true;
  ctx->have_solute = false;
  return RISM3D_OK;
}

static int reset_state(rism3d_ctx* ctx) {
  CU(cudaMemsetAsync(ctx->b.state, 0, sizeof(DevState), ctx->stream));
  CU(cudaMemsetAsync(ctx->b.tickets, 0, ctx->b.n_tickets * sizeof(unsigned), ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_set_solute(rism3d_ctx* ctx, int n_atoms, const double* xyz, const double* q,
                                 const double* sigma, const double* eps, double rcut, float* setup_ms) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (n_atoms < 0 || (n_atoms > 0 && (!xyz || !q || !sigma || !eps))) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  if (!ctx->have_solvent) return fail(ctx, RISM3D_ERR_ORDER, "set_solvent_chi must come before set_solute");
  const Grid& g = ctx->g;
  const SolverParams& sp = ctx->sp;
  const int nv = g.nv;
  // host-side input tables: atom records (x, y, z, beta C q), raw charges, mixed pair parameters
  const size_t na = (size_t)n_atoms;
  std::vector<double> atoms(na * 5), pair(na * nv * 3);
  for (size_t a = 0; a < na; ++a) {
    atoms[4 * a + 0] = xyz[3 * a + 0];
    atoms[4 * a + 1] = xyz[3 * a + 1];
    atoms[4 * a + 2] = xyz[3 * a + 2];
    atoms[4 * a + 3] = sp.beta * COULOMB * q[a];
    atoms[4 * na + a] = q[a];
    for (int s = 0; s < nv; ++s) {
      const double sg = 0.5 * (sigma[a] + ctx->sigv[s]);           // Lorentz-Berthelot (Q4)
      const double ep = sqrt(eps[a] * ctx->epsv[s]);
      pair[(a * nv + s) * 3 + 0] = sp.beta * COULOMB * q[a] * ctx->qv[s];
      pair[(a * nv + s) * 3 + 1] = sg * sg;
      pair[(a * nv + s) * 3 + 2] = 4.0 * sp.beta * ep;
    }
  }
  // With a cutoff the short-range potential comes from a cell list (launch_w_cells): bin the atoms into cubic cells of
  // edge >= rcut / 2 over their bounding box and sort them by cell index (z fastest), host side -- a counting sort of
  // n_atoms records; phi(r), which is never cut off and which the loop never reads, is computed when first needed.
  const bool cells = rcut > 0.0 && n_atoms > 0;
  std::vector<int> cell_start;
  std::vector<double> atoms_s, pair_s, q_s;          // the tables sorted by cell
  int nc[3] = {1, 1, 1};
  double clo[3] = {0.0, 0.0, 0.0}, cedge = rcut > 0.0 ? 0.5 * rcut : 1.0;
  if (cells) {
    double hi[3];
    for (int k = 0; k < 3; ++k) { clo[k] = hi[k] = xyz[k]; }
    for (size_t a = 0; a < na; ++a)
      for (int k = 0; k < 3; ++k) { clo[k] = fmin(clo[k], xyz[3 * a + k]); hi[k] = fmax(hi[k], xyz[3 * a + k]); }
    double span = fmax(hi[0] - clo[0], fmax(hi[1] - clo[1], hi[2] - clo[2]));
    if (!(span < 1e300)) return fail(ctx, RISM3D_ERR_ARG, "non-finite atom coordinates");
    if (span / cedge > 96.0) cedge = span / 96.0;                       // at most ~96 cells per axis
    for (int k = 0; k < 3; ++k) nc[k] = (int)floor((hi[k] - clo[k]) / cedge) + 1;
    const size_t ncell = (size_t)nc[0] * nc[1] * nc[2];
    auto cell_of = [&](size_t a) {
      size_t c[3];
      for (int k = 0; k < 3; ++k) {
        int i = (int)floor((xyz[3 * a + k] - clo[k]) / cedge);
        c[k] = (size_t)(i < 0 ? 0 : (i >= nc[k] ? nc[k] - 1 : i));
      }
      return (c[0] * nc[1] + c[1]) * nc[2] + c[2];
    };
    cell_start.assign(ncell + 1, 0);
    std::vector<size_t> cid(na);
    for (size_t a = 0; a < na; ++a) { cid[a] = cell_of(a); cell_start[cid[a] + 1] += 1; }
    for (size_t c = 0; c < ncell; ++c) cell_start[c + 1] += cell_start[c];
    std::vector<int> fill(cell_start.begin(), cell_start.end() - 1);
    atoms_s.resize(na * 4);
    pair_s.resize(na * nv * 3);
    for (size_t a = 0; a < na; ++a) {                                    // stable: atoms of a cell keep their input order
      const size_t d = (size_t)fill[cid[a]]++;
      for (int k = 0; k < 4; ++k) atoms_s[4 * d + k] = atoms[4 * a + k];
      for (int k = 0; k < nv * 3; ++k) pair_s[d * nv * 3 + k] = pair[a * nv * 3 + k];
    }
    // the sorted tables replace the unsorted ones for the setup kernels of this call (phi~ is a sum over all atoms in
    // any order; its charges follow the atom records); the host copies kept for rism3d_gradient stay in input order
    q_s.resize(na);
    std::vector<int> fill2(cell_start.begin(), cell_start.end() - 1);
    for (size_t a = 0; a < na; ++a) q_s[(size_t)fill2[cid[a]]++] = q[a];
  }
  const std::vector<double>& up_atoms = cells ? atoms_s : atoms;
  const std::vector<double>& up_pair = cells ? pair_s : pair;
  const size_t b_atoms = align256((na * 5) * 8 + 8), b_pair = align256(pair.size() * 8 + 8);
  const size_t b_phase = align256((size_t)3 * na * g.nmax * 16 + 16);
  const size_t b_cells = align256(cell_start.size() * sizeof(int) + 8);
  if (b_atoms + b_pair + b_phase + b_cells > ctx->scratch_bytes)
    return fail(ctx, RISM3D_ERR_WORKSPACE, "%d atoms need %zu scratch bytes, workspace has %zu", n_atoms,
                b_atoms + b_pair + b_phase + b_cells, ctx->scratch_bytes);
  char* scr = (char*)ctx->b.Z;                      // Z, R, tau, w, work are contiguous; the tables live in the
  // history part of the span (rebuilt by the iteration anyway), clear of tau and w, which the setup writes
  const size_t xr_bytes = (size_t)((char*)ctx->b.tau - (char*)ctx->b.Z);
  if (b_atoms + b_pair + b_phase + b_cells > xr_bytes)
    return fail(ctx, RISM3D_ERR_WORKSPACE, "%d atoms need %zu scratch bytes, history span has %zu", n_atoms,
                b_atoms + b_pair + b_phase + b_cells, xr_bytes);
  double* d_atoms = (double*)scr;
  double* d_pair = (double*)(scr + b_atoms);
  double2* d_phase = (double2*)(scr + b_atoms + b_pair);
  int* d_cells = (int*)(scr + b_atoms + b_pair + b_phase);
  ScopedEvents ev;
  CU(ev.create());
  cudaEvent_t e0 = ev.e0, e1 = ev.e1;
  if (na) {
    CU(cudaMemcpyAsync(d_atoms, up_atoms.data(), na * 4 * 8, cudaMemcpyHostToDevice, ctx->stream));
    // raw charges right after the atom records (phi~ reads them there)
    CU(cudaMemcpyAsync(d_atoms + 4 * na, cells ? q_s.data() : atoms.data() + 4 * na, na * 8,
                       cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(d_pair, up_pair.data(), up_pair.size() * 8, cudaMemcpyHostToDevice, ctx->stream));
    if (cells) CU(cudaMemcpyAsync(d_cells, cell_start.data(), cell_start.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
  }
  CU(cudaEventRecord(e0, ctx->stream));
  if (cells) {
    ctx->launches += launch_w_cells(g, ctx->b, sp, d_atoms, d_pair, d_cells, nc, clo, cedge, rcut, ctx->stream);
    ctx->phi_valid = false;
  } else {
    ctx->launches += launch_potential(g, ctx->b, sp, n_atoms, d_atoms, d_pair, rcut, ctx->stream);
    ctx->phi_valid = true;
  }
  CU(cudaGetLastError());
  ctx->launches += launch_phi_tilde(g, ctx->b, sp, n_atoms, d_atoms, d_phase, ctx->stream);
  CU(cudaGetLastError());
  CU(cudaEventRecord(e1, ctx->stream));
  // tau = 0 (t = f); empty history
  CU(cudaMemsetAsync(ctx->b.tau, 0, g.field * 8, ctx->stream));
  int rc = reset_state(ctx);
  if (rc) return rc;
  CU(cudaStreamSynchronize(ctx->stream));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  if (setup_ms) *setup_ms = ms;
  if (!ctx->h_atoms) ctx->h_atoms = new std::vector<double>();
  if (!ctx->h_pair) ctx->h_pair = new std::vector<double>();
  ctx->h_atoms->assign(atoms.begin(), atoms.begin() + 4 * na);
  *ctx->h_pair = pair;
  ctx->n_atoms = n_atoms;
  ctx->phi_ms = 0.f;
  ctx->have_solute = true;
  return RISM3D_OK;
}

__global__ void iterate_begin_kernel(DevState* st, double tol) {
  st->tol = tol;
  st->done = 0;
  st->status = 0;
  st->n_done = 0;
}

// profiling: one event before the first loop kernel and one after each (RISM3D_N_LOOP_KERNELS + 1 per iteration)
static void prof_mark(rism3d_ctx* ctx) {
  if (!ctx->profiling) return;
  if (!ctx->ev_pool) ctx->ev_pool = new std::vector<cudaEvent_t>();
  if (ctx->ev_used == ctx->ev_pool->size()) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) { ctx->profiling = false; return; }
    ctx->ev_pool->push_back(e);
  }
  cudaEventRecord((*ctx->ev_pool)[ctx->ev_used++], ctx->stream);
}

// after the stream has been synchronised: fold the recorded events into the per-kernel sums
static void prof_collect(rism3d_ctx* ctx) {
  if (!ctx->ev_pool) return;
  const size_t per = RISM3D_N_LOOP_KERNELS + 1;
  for (size_t i = 0; i + per <= ctx->ev_used; i += per) {
    for (int k = 0; k < RISM3D_N_LOOP_KERNELS; ++k) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, (*ctx->ev_pool)[i + k], (*ctx->ev_pool)[i + k + 1]) == cudaSuccess)
        ctx->prof_ms[k] += ms;
    }
    ctx->prof_iters += 1;
  }
  ctx->ev_used = 0;
}

constexpr int GRAPH_PACK = 8;   // iterations per large graph = iterations between two convergence checks of iterate

static int enqueue_iteration(rism3d_ctx* ctx) {
  const Grid& g = ctx->g;
  const Buffers& b = ctx->b;
  cudaStream_t s = ctx->stream;
  const bool peers = g.n_ranks > 1;                        // (rism3d_iterate only gets here in peer mode)
  int k = 0;
  prof_mark(ctx);
  k += launch_closure_zfwd(g, b, ctx->sp, nullptr, s);     // step 2 + z of step 3
  prof_mark(ctx);
  k += launch_y_fwd(g, b, true, s);                        // step 3 (slab run: stores into the peers' k-space slabs)
  if (peers) k += launch_xbarrier(g, b, s);
  prof_mark(ctx);
  k += launch_kspace_x(g, b, s);                           // step 3 (x), Eq. 32, step 4, x of step 5
  if (peers) k += launch_xbarrier(g, b, s);
  prof_mark(ctx);
  k += launch_y_inv(g, b, true, s);                        // step 5 (slab run: loads from the peers' k-space slabs)
  prof_mark(ctx);
  k += launch_zinv_residual(g, b, ctx->sp, nullptr, s);    // step 5 (z), Eq. 33, steps 6-7: Gram row, rms test, MDIIS solve
  if (peers) {
    k += launch_xbarrier(g, b, s);                         // every rank's Gram row has arrived; nobody reads K any more
    k += launch_gram_solve(g, b, ctx->sp, s);
  }
  prof_mark(ctx);                                          // (the update tau = sum c_i Z_i is applied by the next
                                                           //  closure_zfwd, or by iterate's trailing update pass)
  ctx->launches += k;
  return k;
}

// capture `iters` iterations into an executable graph; nullptr when capture is not possible on this stream
static cudaGraphExec_t capture_iterations(rism3d_ctx* ctx, int iters, int* kernels_per_iteration) {
  if (cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  const long long before = ctx->launches;
  int k = 0;
  for (int i = 0; i < iters; ++i) k = enqueue_iteration(ctx);
  ctx->launches = before;                                  // captured, not launched
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  if (cudaStreamEndCapture(ctx->stream, &graph) != cudaSuccess || graph == nullptr) {
    cudaGetLastError();
    return nullptr;
  }
  if (cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    cudaGetLastError();
    exec = nullptr;
  }
  cudaGraphDestroy(graph);
  if (kernels_per_iteration) *kernels_per_iteration = k;
  return exec;
}

// enqueue `iters` (1 or GRAPH_PACK) iterations: as a graph launch when possible, else kernel by kernel
static void enqueue_iterations(rism3d_ctx* ctx, int iters) {
  if (!ctx->profiling && ctx->stream != nullptr) {
    if (!ctx->graph_tried) {
      ctx->graph_tried = true;
      int k = 0;
      ctx->graph1 = capture_iterations(ctx, 1, &k);
      ctx->graph_pack = ctx->graph1 ? capture_iterations(ctx, GRAPH_PACK, &k) : nullptr;
      ctx->graph_kernels = k;
    }
    cudaGraphExec_t exec = (iters == GRAPH_PACK) ? ctx->graph_pack : (iters == 1 ? ctx->graph1 : nullptr);
    if (exec && cudaGraphLaunch(exec, ctx->stream) == cudaSuccess) {
      ctx->launches += (long long)ctx->graph_kernels * iters;
      return;
    }
  }
  for (int i = 0; i < iters; ++i) enqueue_iteration(ctx);
}

extern "C" int rism3d_set_profiling(rism3d_ctx* ctx, int enable) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  CU(cudaStreamSynchronize(ctx->stream));
  ctx->ev_used = 0;
  ctx->profiling = enable != 0;
  for (int k = 0; k < RISM3D_N_LOOP_KERNELS; ++k) ctx->prof_ms[k] = 0.0;
  ctx->prof_iters = 0;
  return RISM3D_OK;
}

extern "C" int rism3d_get_timings(rism3d_ctx* ctx, double* ms_total, int cap, long long* n_iterations) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!ms_total || cap < RISM3D_N_LOOP_KERNELS) return fail(ctx, RISM3D_ERR_ARG, "ms_total needs %d entries", RISM3D_N_LOOP_KERNELS);
  CU(cudaStreamSynchronize(ctx->stream));
  prof_collect(ctx);
  for (int k = 0; k < RISM3D_N_LOOP_KERNELS; ++k) ms_total[k] = ctx->prof_ms[k];
  if (n_iterations) *n_iterations = ctx->prof_iters;
  return RISM3D_OK;
}

extern "C" const char* rism3d_loop_kernel_name(int k) {
  static const char* names[RISM3D_N_LOOP_KERNELS] = {"closure_zfwd", "y_fwd", "kspace_x", "y_inv", "zinv_gram_solve"};
  return (k >= 0 && k < RISM3D_N_LOOP_KERNELS) ? names[k] : "";
}

static int read_header(rism3d_ctx* ctx) {
  CU(cudaMemcpyAsync(ctx->h_hdr, ctx->b.state, sizeof(StateHeader), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_iterate(rism3d_ctx* ctx, int max_iter, double tol, int* n_done, double* rms) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (max_iter < 0) return fail(ctx, RISM3D_ERR_ARG, "max_iter < 0");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before iterate");
  if (ctx->g.n_ranks > 1 && !ctx->b.peer_mode)
    return fail(ctx, RISM3D_ERR_ORDER, "a staged slab run is driven by rism3d_slab_phase (or call rism3d_slab_set_peers)");
  if (ctx->peer_broken)
    return fail(ctx, RISM3D_ERR_PEER, "an earlier iterate gave up at an in-stream barrier: the ranks' barrier epochs no longer "
                                      "agree; call rism3d_slab_set_peers on every rank (then a host-side barrier) first");
  iterate_begin_kernel<<<1, 1, 0, ctx->stream>>>(ctx->b.state, tol);
  ctx->launches += 1;
  // packs of GRAPH_PACK iterations (one graph launch each) with a look at the device state in between when a
  // tolerance is set; once an iteration has converged the remaining kernels of a pack return immediately
  int it = 0;
  while (it < max_iter) {
    const int step = (max_iter - it >= GRAPH_PACK) ? GRAPH_PACK : 1;
    enqueue_iterations(ctx, step);
    it += step;
    if (tol > 0.0 && step == GRAPH_PACK) {
      int rc = read_header(ctx);
      if (rc) return rc;
      if (ctx->h_hdr->done) break;
    }
  }
  // the update of the last iteration is still pending (it rides on the next closure pass): apply it now, so that
  // tau is the new input when this call returns
  if (max_iter > 0) ctx->launches += launch_mdiis_update(ctx->g, ctx->b, ctx->sp, ctx->stream);
  CU(cudaGetLastError());
  int rc = read_header(ctx);
  if (rc) return rc;
  prof_collect(ctx);
  if (n_done) *n_done = ctx->h_hdr->n_done;
  if (rms) *rms = ctx->h_hdr->rms_last;
  if (ctx->h_hdr->status == RISM3D_ERR_DIVERGED)
    return fail(ctx, RISM3D_ERR_DIVERGED, "non-finite residual after %d iterations", ctx->h_hdr->n_done);
  if (ctx->h_hdr->status == RISM3D_ERR_PEER) {
    ctx->peer_broken = true;
    return fail(ctx, RISM3D_ERR_PEER, "a peer rank did not reach an in-stream barrier within %.3g s (after %d iterations): "
                "the iteration was abandoned on this rank", (double)ctx->b.peer_timeout_ns * 1e-9, ctx->h_hdr->n_done);
  }
  return RISM3D_OK;
}

// phi(r) of the current solute, computed on first use when set_solute took the cell-list path (the loop never reads
// phi; the free energy and the T / PHI getters do).  The atom table goes through the k-space work array, which holds
// nothing between iterations.
static int ensure_phi(rism3d_ctx* ctx) {
  if (ctx->phi_valid) return RISM3D_OK;
  const size_t na = (size_t)ctx->n_atoms;
  if (na * 4 * 8 > ctx->g.field * 8) return fail(ctx, RISM3D_ERR_WORKSPACE, "%d atoms do not fit the work array", ctx->n_atoms);
  double* d_atoms = (double*)ctx->b.work;
  ScopedEvents ev;
  CU(ev.create());
  cudaEvent_t e0 = ev.e0, e1 = ev.e1;
  CU(cudaMemcpyAsync(d_atoms, ctx->h_atoms->data(), na * 4 * 8, cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaEventRecord(e0, ctx->stream));
  ctx->launches += launch_phi(ctx->g, ctx->b, ctx->sp, ctx->n_atoms, d_atoms, ctx->stream);
  CU(cudaGetLastError());
  CU(cudaEventRecord(e1, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  CU(cudaEventElapsedTime(&ctx->phi_ms, e0, e1));
  ctx->phi_valid = true;
  return RISM3D_OK;
}

extern "C" int rism3d_measure_dfma_peak(rism3d_ctx* ctx, double* tflops) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!tflops) return fail(ctx, RISM3D_ERR_ARG, "tflops is NULL");
  CU(cudaStreamSynchronize(ctx->stream));
  *tflops = measure_dfma_peak(ctx->g.num_sms, ctx->d_out, ctx->stream);
  ctx->launches += 5;
  CU(cudaGetLastError());
  return RISM3D_OK;
}

extern "C" int rism3d_phi_ms(rism3d_ctx* ctx, float* ms) {
  if (!ctx) return RISM3D_ERR_ARG;
  if (!ms) return fail(ctx, RISM3D_ERR_ARG, "ms is NULL");
  *ms = ctx->phi_valid ? ctx->phi_ms : 0.f;
  return RISM3D_OK;
}

extern "C" int rism3d_free_energy(rism3d_ctx* ctx, double* dmu_total, double* dmu_site) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!dmu_total) return fail(ctx, RISM3D_ERR_ARG, "dmu_total is NULL");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before free_energy");
  { const int rc_phi = ensure_phi(ctx); if (rc_phi) return rc_phi; }
  ctx->launches += launch_free_energy(ctx->g, ctx->b, ctx->sp, ctx->d_out, ctx->stream);
  CU(cudaGetLastError());
  double host[MAX_NV];
  CU(cudaMemcpyAsync(host, ctx->d_out, ctx->g.nv * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  double tot = 0.0;
  for (int i = 0; i < ctx->g.nv_user; ++i) {
    tot += host[i];
    if (dmu_site) dmu_site[i] = host[i];
  }
  *dmu_total = tot;
  return RISM3D_OK;
}

extern "C" int rism3d_pmv(rism3d_ctx* ctx, double chi_t, double* pmv, double* c_int_site) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!pmv) return fail(ctx, RISM3D_ERR_ARG, "pmv is NULL");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before pmv");
  { const int rc_phi = ensure_phi(ctx); if (rc_phi) return rc_phi; }
  ctx->launches += launch_free_energy(ctx->g, ctx->b, ctx->sp, ctx->d_out, ctx->stream);
  CU(cudaGetLastError());
  double host[2 * MAX_NV];
  CU(cudaMemcpyAsync(host, ctx->d_out, 2 * MAX_NV * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  double sum = 0.0;                                  // sum_g rho_g int c_g dr: the -q_g phi part drops out (sum rho q = 0)
  for (int i = 0; i < ctx->g.nv_user; ++i) {
    sum += ctx->rhov[i] * host[MAX_NV + i];
    if (c_int_site) c_int_site[i] = host[MAX_NV + i];
  }
  *pmv = ctx->sp.kT * chi_t * ((ctx->g.rank == 0 ? 1.0 : 0.0) - sum);   // Eq. 19 (slab run: this slab's share)
  return RISM3D_OK;
}

extern "C" int rism3d_pressure_correction(rism3d_ctx* ctx, double chi_t, double pressure, double* dmu_pc, double* pmv) {
  if (!ctx) return RISM3D_ERR_ARG;
  if (!dmu_pc) return fail(ctx, RISM3D_ERR_ARG, "dmu_pc is NULL");
  double v = 0.0;
  const int rc = rism3d_pmv(ctx, chi_t, &v, nullptr);     // Eq. 19
  if (rc) return rc;
  *dmu_pc = -pressure * v;                                 // Eq. 21
  if (pmv) *pmv = v;
  return RISM3D_OK;
}

extern "C" int rism3d_gradient(rism3d_ctx* ctx, double* grad) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!grad) return fail(ctx, RISM3D_ERR_ARG, "grad is NULL");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before gradient");
  const Grid& g = ctx->g;
  const int na = ctx->n_atoms;
  if (na == 0) return RISM3D_OK;
  // Scratch: the k-space work array (nothing lives there between iterations) takes rho dV g; the history slot `cur`
  // that the NEXT (Z, R) pair will overwrite -- an unused slot, or the oldest entry, which the trailing update of
  // iterate has already consumed and the next Gram row skips -- takes the tables, the partial sums and the result.
  int rc = read_header(ctx);
  if (rc) return rc;
  const int cur = ctx->h_hdr->cur;
  const size_t b_atoms = align256((size_t)na * 4 * 8), b_pair = align256((size_t)na * g.nv * 3 * 8);
  const size_t b_out = align256((size_t)na * 3 * 8);
  const size_t avail = g.field * 8;
  if (b_atoms + b_pair + b_out + (size_t)na * 3 * 16 > avail)
    return fail(ctx, RISM3D_ERR_WORKSPACE, "%d atoms do not fit one field-set of scratch on this grid", na);
  size_t nchunks = (g.npts + 8191) / 8192;                 // >= 8192 points per block, fewer blocks if memory is short
  const size_t max_chunks = (avail - b_atoms - b_pair - b_out) / ((size_t)na * 3 * 16);
  if (nchunks > max_chunks) nchunks = max_chunks;
  if (nchunks > 2048) nchunks = 2048;
  char* base = (char*)(ctx->b.R + (size_t)cur * g.field);
  double* d_atoms = (double*)base;
  double* d_pair = (double*)(base + b_atoms);
  double* d_out = (double*)(base + b_atoms + b_pair);
  double* d_part = (double*)(base + b_atoms + b_pair + b_out);
  CU(cudaMemcpyAsync(d_atoms, ctx->h_atoms->data(), (size_t)na * 4 * 8, cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaMemcpyAsync(d_pair, ctx->h_pair->data(), (size_t)na * g.nv * 3 * 8, cudaMemcpyHostToDevice, ctx->stream));
  ctx->launches += launch_gradient(g, ctx->b, ctx->sp, na, (double*)ctx->b.work, d_atoms, d_pair, d_part, (int)nchunks,
                                   d_out, ctx->stream);
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(grad, d_out, (size_t)na * 3 * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_get_field(rism3d_ctx* ctx, int which, int site, double* dst, int dst_is_device) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!dst || which < 0 || which > RISM3D_FIELD_PHI || site < 0 || site >= ctx->g.nv_user)
    return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before get_field");
  if (which == RISM3D_FIELD_T || which == RISM3D_FIELD_PHI) { const int rc_phi = ensure_phi(ctx); if (rc_phi) return rc_phi; }
  double* d = dst_is_device ? dst : ctx->b.scratch;
  ctx->launches += launch_get_field(ctx->g, ctx->b, ctx->sp, which, site, d, ctx->stream);
  CU(cudaGetLastError());
  if (!dst_is_device) CU(cudaMemcpyAsync(dst, d, ctx->g.npts * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_set_tau(rism3d_ctx* ctx, int site, const double* src, int src_is_device) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!src || site < 0 || site >= ctx->g.nv_user) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before set_tau");
  const Grid& g = ctx->g;
  CU(cudaMemcpyAsync(ctx->b.tau + (size_t)site * g.npts, src, g.npts * 8,
                     src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
  int rc;
  rc = reset_state(ctx);
  if (rc) return rc;
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_get_rms_history(rism3d_ctx* ctx, double* dst, int cap, int* n) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!dst || cap < 0 || !n) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  int rc = read_header(ctx);
  if (rc) return rc;
  int total = ctx->h_hdr->hist_n;
  int avail = total < RMS_HIST_CAP ? total : RMS_HIST_CAP;
  int cnt = avail < cap ? avail : cap;
  std::vector<double> tmp(RMS_HIST_CAP);
  CU(cudaMemcpyAsync(tmp.data(), (char*)ctx->b.state + offsetof(DevState, rms_hist), (size_t)RMS_HIST_CAP * 8,
                     cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int i = 0; i < cnt; ++i) dst[i] = tmp[(size_t)(total - cnt + i) % RMS_HIST_CAP];
  *n = cnt;
  return RISM3D_OK;
}

extern "C" int rism3d_slab_plan(const rism3d_params* p, rism3d_slab_info* out) {
  if (!p || !out) return RISM3D_ERR_ARG;
  if (!valid_params(p)) return RISM3D_ERR_SIZE;
  const Grid g = make_grid(p);
  out->nxl = g.nxl; out->ix0 = g.ix0; out->nyl = g.nyl; out->jy0 = g.jy0;
  out->n_sites_padded = g.nv;
  out->row_elems = g.q();
  out->block_elems = (size_t)g.nxl * g.nyl * g.q();
  return RISM3D_OK;
}

// ---- slab decomposition: exchange addresses, peer tables, phase calls (include/rism3d.h "Slab decomposition") ----
extern "C" int rism3d_slab_local(rism3d_ctx* ctx, void** d_K, void** d_stage, void** d_gram, void** d_flags,
                                 size_t* block_bytes, size_t* gram_row_bytes) {
  if (!ctx) return RISM3D_ERR_ARG;
  const Grid& g = ctx->g;
  if (g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  if (d_K) *d_K = ctx->b.kbuf;
  if (d_stage) *d_stage = ctx->b.stage;
  if (d_gram) *d_gram = ctx->b.gram_x;
  if (d_flags) *d_flags = ctx->b.xflags;
  if (block_bytes) *block_bytes = (size_t)g.nxl * g.nyl * g.q() * sizeof(double2);
  if (gram_row_bytes) *gram_row_bytes = (size_t)GRAM_SLOT * 2 * sizeof(double);
  return RISM3D_OK;
}

extern "C" int rism3d_slab_set_peers(rism3d_ctx* ctx, void* const* d_K, void* const* d_gram, void* const* d_flags) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  Grid& g = ctx->g;
  if (g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  if (!d_K || !d_gram || !d_flags) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  for (int r = 0; r < g.n_ranks; ++r)
    if (!d_K[r] || !d_gram[r] || !d_flags[r]) return fail(ctx, RISM3D_ERR_ARG, "peer %d: NULL pointer", r);
  if (d_K[g.rank] != (void*)ctx->b.kbuf || d_gram[g.rank] != (void*)ctx->b.gram_x || d_flags[g.rank] != (void*)ctx->b.xflags)
    return fail(ctx, RISM3D_ERR_ARG, "entry %d must be this rank's own arrays (rism3d_slab_local)", g.rank);
  // every (re)connection starts the barrier epochs from zero on every rank: a rank whose context was re-created would
  // otherwise count from 0 while the others keep their old epochs (all ranks call set_peers, then meet on the host)
  CU(cudaMemsetAsync(ctx->b.xflags, 0, (MAX_RANKS + 1) * sizeof(unsigned long long), ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  ctx->peer_broken = false;
  // rank r's rows of the spectrum sit in block `rank` of rank r's K: stores on the way in, loads on the way out
  const size_t blk = (size_t)g.nxl * g.nyl * g.q();
  for (int r = 0; r < g.n_ranks; ++r) {
    ctx->b.fwd_dst[r] = (double2*)d_K[r] + (size_t)g.rank * blk;
    ctx->b.bwd_src[r] = (const double2*)d_K[r] + (size_t)g.rank * blk;
    ctx->b.gram_dst[r] = (double*)d_gram[r];
    ctx->b.flag_dst[r] = (unsigned long long*)d_flags[r];
  }
  ctx->b.n_gram_dst = g.n_ranks;
  ctx->b.peer_mode = true;
  // graphs captured before the switch hold the old tables
  if (ctx->graph1) { cudaGraphExecDestroy(ctx->graph1); ctx->graph1 = nullptr; }
  if (ctx->graph_pack) { cudaGraphExecDestroy(ctx->graph_pack); ctx->graph_pack = nullptr; }
  ctx->graph_tried = false;
  return RISM3D_OK;
}

extern "C" int rism3d_slab_combine(const double* per_rank, int n_ranks, int n_values, double* out) {
  if (!per_rank || !out || n_ranks < 1 || n_ranks > MAX_RANKS || n_values < 0) return RISM3D_ERR_ARG;
  for (int j = 0; j < n_values; ++j) {
    double acc = 0.0;
    for (int r = 0; r < n_ranks; ++r) acc += per_rank[(size_t)r * n_values + j];   // fixed rank order, as the Gram rows
    out[j] = acc;
  }
  return RISM3D_OK;
}

extern "C" int rism3d_slab_set_peer_timeout(rism3d_ctx* ctx, double seconds) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (ctx->g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  if (!(seconds >= 1e-3) || !(seconds <= 3600.0)) return fail(ctx, RISM3D_ERR_ARG, "timeout %g s outside 0.001..3600", seconds);
  CU(cudaStreamSynchronize(ctx->stream));
  ctx->b.peer_timeout_ns = (unsigned long long)(seconds * 1e9);
  // the limit is a launch parameter of the captured barrier kernels
  if (ctx->graph1) { cudaGraphExecDestroy(ctx->graph1); ctx->graph1 = nullptr; }
  if (ctx->graph_pack) { cudaGraphExecDestroy(ctx->graph_pack); ctx->graph_pack = nullptr; }
  ctx->graph_tried = false;
  return RISM3D_OK;
}

extern "C" int rism3d_debug_peer_barrier_selftest(int device, void* d_scratch, size_t bytes, void* cuda_stream, int n_ranks,
                                                  int epochs, int absent_rank, double timeout_s, int* n_errors,
                                                  int* n_timeouts) {
  if (!d_scratch || bytes < 4096 || !n_errors || !n_timeouts) return RISM3D_ERR_ARG;
  if (n_ranks < 1 || n_ranks > MAX_RANKS || epochs < 1 || absent_rank >= n_ranks) return RISM3D_ERR_ARG;
  if (!(timeout_s >= 1e-3) || !(timeout_s <= 60.0)) return RISM3D_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return RISM3D_ERR_CUDA;
  DeviceGuard guard(device);
  int res[2] = {-1, -1};
  if (run_xbarrier_selftest(d_scratch, n_ranks, epochs, absent_rank, (unsigned long long)(timeout_s * 1e9), res,
                            (cudaStream_t)cuda_stream) != cudaSuccess) {
    cudaGetLastError();
    return RISM3D_ERR_CUDA;
  }
  *n_errors = res[0];
  *n_timeouts = res[1];
  return RISM3D_OK;
}

// ---- CUDA IPC helpers for peer mode ----
static_assert(sizeof(cudaIpcMemHandle_t) == 64, "the ABI passes IPC handles as 64 bytes");

extern "C" int rism3d_peer_alloc(int device, size_t bytes, void** d_ptr) {
  if (!d_ptr || bytes == 0) return RISM3D_ERR_ARG;
  if (!device_exists(device)) return RISM3D_ERR_ARG;
  DeviceGuard guard(device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  return cudaMalloc(d_ptr, bytes) == cudaSuccess ? RISM3D_OK : RISM3D_ERR_CUDA;
}

extern "C" int rism3d_peer_free(int device, void* d_ptr) {
  if (!device_exists(device)) return RISM3D_ERR_ARG;
  DeviceGuard guard(device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  return cudaFree(d_ptr) == cudaSuccess ? RISM3D_OK : RISM3D_ERR_CUDA;
}

extern "C" int rism3d_peer_export(int device, void* d_ptr, unsigned char handle[64]) {
  if (!d_ptr || !handle) return RISM3D_ERR_ARG;
  if (!device_exists(device)) return RISM3D_ERR_ARG;
  DeviceGuard guard(device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  cudaIpcMemHandle_t h;
  if (cudaIpcGetMemHandle(&h, d_ptr) != cudaSuccess) return RISM3D_ERR_CUDA;
  memcpy(handle, &h, 64);
  return RISM3D_OK;
}

extern "C" int rism3d_peer_open(int device, const unsigned char handle[64], void** d_ptr) {
  if (!d_ptr || !handle) return RISM3D_ERR_ARG;
  if (!device_exists(device)) return RISM3D_ERR_ARG;
  DeviceGuard guard(device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle, 64);
  return cudaIpcOpenMemHandle(d_ptr, h, cudaIpcMemLazyEnablePeerAccess) == cudaSuccess ? RISM3D_OK : RISM3D_ERR_CUDA;
}

extern "C" int rism3d_peer_close(int device, void* d_ptr) {
  if (!device_exists(device)) return RISM3D_ERR_ARG;
  DeviceGuard guard(device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  return cudaIpcCloseMemHandle(d_ptr) == cudaSuccess ? RISM3D_OK : RISM3D_ERR_CUDA;
}

extern "C" int rism3d_slab_begin(rism3d_ctx* ctx, double tol) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (ctx->g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before the iteration");
  iterate_begin_kernel<<<1, 1, 0, ctx->stream>>>(ctx->b.state, tol);
  ctx->launches += 1;
  CU(cudaGetLastError());
  return RISM3D_OK;
}

extern "C" int rism3d_slab_phase(rism3d_ctx* ctx, int phase) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  const Grid& g = ctx->g;
  if (g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  if (!ctx->have_solute) return fail(ctx, RISM3D_ERR_ORDER, "set_solute must come before the iteration");
  cudaStream_t s = ctx->stream;
  int k = 0;
  switch (phase) {
    case 0:
      k += launch_closure_zfwd(g, ctx->b, ctx->sp, nullptr, s);
      k += launch_y_fwd(g, ctx->b, true, s);
      break;
    case 1: k += launch_kspace_x(g, ctx->b, s); break;
    case 2:
      k += launch_y_inv(g, ctx->b, true, s);
      k += launch_zinv_residual(g, ctx->b, ctx->sp, nullptr, s);
      break;
    case 3: k += launch_gram_solve(g, ctx->b, ctx->sp, s); break;
    default: return fail(ctx, RISM3D_ERR_ARG, "phase %d (0..3)", phase);
  }
  ctx->launches += k;
  CU(cudaGetLastError());
  return RISM3D_OK;
}

extern "C" int rism3d_slab_status(rism3d_ctx* ctx, int* done, int* n_done, double* rms) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  int rc = read_header(ctx);
  if (rc) return rc;
  if (done) *done = ctx->h_hdr->done;
  if (n_done) *n_done = ctx->h_hdr->n_done;
  if (rms) *rms = ctx->h_hdr->rms_last;
  return RISM3D_OK;
}

extern "C" int rism3d_slab_end(rism3d_ctx* ctx, int* n_done, double* rms) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (ctx->g.n_ranks <= 1) return fail(ctx, RISM3D_ERR_ORDER, "not a slab run (rism3d_params.n_ranks <= 1)");
  ctx->launches += launch_mdiis_update(ctx->g, ctx->b, ctx->sp, ctx->stream);   // no-op when nothing is pending
  CU(cudaGetLastError());
  int rc = read_header(ctx);
  if (rc) return rc;
  if (n_done) *n_done = ctx->h_hdr->n_done;
  if (rms) *rms = ctx->h_hdr->rms_last;
  if (ctx->h_hdr->status == RISM3D_ERR_DIVERGED)
    return fail(ctx, RISM3D_ERR_DIVERGED, "non-finite residual after %d iterations", ctx->h_hdr->n_done);
  return RISM3D_OK;
}

extern "C" int rism3d_debug_fft_forward(rism3d_ctx* ctx, const double* d_in, double* d_out) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!d_in || !d_out) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  const Grid& g = ctx->g;
  if (g.n_ranks > 1) return fail(ctx, RISM3D_ERR_ORDER, "the debug transforms are single-rank only");
  int k = launch_closure_zfwd(g, ctx->b, ctx->sp, d_in, ctx->stream);
  k += launch_y_fwd(g, ctx->b, false, ctx->stream);
  k += launch_x_fwd(g, ctx->b, ctx->stream);
  ctx->launches += k;
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(d_out, ctx->b.work, g.field * 8, cudaMemcpyDeviceToDevice, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism3d_debug_fft_inverse(rism3d_ctx* ctx, const double* d_in, double* d_out) {
  if (!ctx) return RISM3D_ERR_ARG;
  ON_CTX_DEVICE(ctx);
  if (!d_in || !d_out) return fail(ctx, RISM3D_ERR_ARG, "bad argument");
  const Grid& g = ctx->g;
  if (g.n_ranks > 1) return fail(ctx, RISM3D_ERR_ORDER, "the debug transforms are single-rank only");
  CU(cudaMemcpyAsync(ctx->b.work, d_in, g.field * 8, cudaMemcpyDeviceToDevice, ctx->stream));
  int k = launch_x_inv(g, ctx->b, ctx->stream);
  k += launch_y_inv(g, ctx->b, false, ctx->stream);
  k += launch_zinv_residual(g, ctx->b, ctx->sp, d_out, ctx->stream);
  ctx->launches += k;
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}
