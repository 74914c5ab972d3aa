// api.cu -- the C-ABI of include/lqcd.h: argument checks, geometry, solver drivers.  No compute here
// beyond launching the kernels of dw.cu / clover.cu / layout.cu / blas.cu; there is no CPU fallback.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <chrono>
#include <mutex>
#include <vector>

#include "cg.cuh"

namespace lqcd {

static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches(0);

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  set_error("%s: %s", what, cudaGetErrorString(e));
  return false;
}
void count_launch(int n) { g_launches += n; }

// lqcd_set_option("host_slab", n): time slices per staged gauge slab of lqcd_dw_apply_host (0 = automatic); takes
// effect when the cached host context is next rebuilt
static int g_host_slab_opt = 0;
static bool g_host_slab_changed = false;
void set_host_slab(int n) { g_host_slab_changed = g_host_slab_changed || n != g_host_slab_opt; g_host_slab_opt = n; }

static int ilog2(int v) {
  int l = 0;
  while ((1 << l) < v) l++;
  return l;
}

// largest power of two <= cap that divides L
static int pow2_divisor(int L, int cap) {
  int b = 1;
  while (b * 2 <= cap && L % (b * 2) == 0) b *= 2;
  return b;
}

static bool parse_ints(const char* s, int* out, int n) {
  if (!s) return false;
  for (int i = 0; i < n; i++) {
    char* end;
    long v = strtol(s, &end, 10);
    if (end == s) return false;
    out[i] = (int)v;
    s = end;
    if (*s == ',' || *s == 'x') s++;
  }
  return true;
}

// Tile shape: 4x4x4x4 sites (TV = 128 per parity, 256 threads for the full operator) when the extents allow
// it, else 8x4x4x2; smaller powers of two otherwise; a longer time extent of the tile when the spatial one is short.
static void choose_tiling(Geom& g) {
  int b[4];
  b[0] = pow2_divisor(g.L[0], 8);
  b[1] = pow2_divisor(g.L[1], 4);
  b[2] = pow2_divisor(g.L[2], 4);
  b[3] = 2;
  if (g.L[0] % 4 == 0 && g.L[1] % 4 == 0 && g.L[2] % 4 == 0 && g.L[3] % 4 == 0) {
    // 4^4: the smallest surface (512 halo sites per 256) and four equal faces, which is what lets the
    // double-buffered halo area of the persistent kernel fit shared memory in fp64
    b[0] = b[1] = b[2] = b[3] = 4;
  }
  int env[4];
  if (parse_ints(getenv("LQCD_TILE"), env, 4)) {
    bool ok = true;
    for (int i = 0; i < 4; i++)
      ok = ok && env[i] >= 2 && (env[i] & (env[i] - 1)) == 0 && g.L[i] % env[i] == 0;
    if (ok && (env[0] / 2) * env[1] * env[2] * env[3] <= 128)
      for (int i = 0; i < 4; i++) b[i] = env[i];
  } else {
    while ((b[0] / 2) * b[1] * b[2] * b[3] < 128 && g.L[3] % (b[3] * 2) == 0 && b[3] < 8) b[3] *= 2;
  }
  for (int i = 0; i < 4; i++) {
    g.b[i] = b[i];
    g.nt[i] = g.L[i] / b[i];
  }
  g.lb[0] = ilog2(b[0] / 2);
  for (int i = 1; i < 4; i++) g.lb[i] = ilog2(b[i]);
  g.TV = (b[0] / 2) * b[1] * b[2] * b[3];
  g.ntiles = g.nt[0] * g.nt[1] * g.nt[2] * g.nt[3];
  // L2 chunking: sweep direction sw inside a chunk of (c1 x c2) tiles along (da, db) so that one layer of the chunk
  // (the reuse distance of a neighbour in the sweep direction) stays well inside L2.  Chunk borders cut the faces of da
  // and db: a cut face is gathered from DRAM a second time, in whole 128-byte lines.  With the site order inside a
  // tile (lqcd_internal.cuh) the x3 and x4 faces are contiguous runs of >= 128 bytes while an x2 face uses a quarter of
  // every line it touches, so the default sweeps x2 (direction 1) and chunks (x3, x4); cut as few faces as possible.
  int sw = 1;
  if (getenv("LQCD_SWEEP")) {
    const int e = atoi(getenv("LQCD_SWEEP"));
    if (e >= 1 && e <= 3) sw = e;
  }
  g.sw = sw;
  g.da = sw == 1 ? 2 : 1;
  g.db = sw == 3 ? 2 : 3;
  long budget = 32768;
  if (getenv("LQCD_LAYER_SITES")) budget = atol(getenv("LQCD_LAYER_SITES"));
  int best1 = 1, best2 = 1;
  double best_cost = 1e30;
  long best_sites = 0;
  const int na = g.nt[g.da], nb = g.nt[g.db];
  for (int c1 = 1; c1 <= na; c1++) {
    if (na % c1) continue;
    for (int c2 = 1; c2 <= nb; c2++) {
      if (nb % c2) continue;
      long sites = (long)g.L[0] * c1 * b[g.da] * c2 * b[g.db] * b[sw];
      if (sites > budget && !(c1 == 1 && c2 == 1)) continue;
      double cost = (c1 < na ? 1.0 / (c1 * b[g.da]) : 0.0) + (c2 < nb ? 1.0 / (c2 * b[g.db]) : 0.0);
      if (cost < best_cost - 1e-12 || (fabs(cost - best_cost) <= 1e-12 && sites > best_sites)) {
        best_cost = cost; best_sites = sites; best1 = c1; best2 = c2;
      }
    }
  }
  int ce[2];
  if (parse_ints(getenv("LQCD_CHUNK"), ce, 2) && ce[0] >= 1 && ce[1] >= 1 && na % ce[0] == 0 && nb % ce[1] == 0) {
    best1 = ce[0]; best2 = ce[1];
  }
  g.c1 = best1;
  g.c2 = best2;
}

static cudaStream_t as_stream(void* s) { return (cudaStream_t)s; }

static size_t spinor_complex(const Geom& g) { return (size_t)2 * g.Vh * 12; }
static size_t elem_bytes(lqcd_prec p) { return p == LQCD_F64 ? sizeof(double2) : sizeof(float2); }
// Length of the per-CTA partial-sum buffer: the largest grid any reducing kernel can have on this geometry --
// 2 * ntiles (dw_mode = split: one CTA per tile parity), sm_count * 8 resident CTAs (persistent one-thread-per-site
// kernels: at most 8 CTAs of >= 128 threads with > 64 registers fit an SM), two values per CTA of the BLAS-1 kernels
// (dot: re and im; grid <= 8 CTAs per SM) -- plus 64 doubles of scratch at the end.
static size_t partial_len(const Geom& g) {
  size_t n = (size_t)2 * g.ntiles;
  const size_t r = (size_t)2 * 8 * (g.sm_count > 0 ? g.sm_count : 148);
  if (r > n) n = r;
  return n + 64;
}
static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool valid_prec(lqcd_prec p) { return p == LQCD_F64 || p == LQCD_F32; }
static bool valid_recon(lqcd_recon r) { return r == LQCD_RECON_18 || r == LQCD_RECON_12; }

// workspace carving
struct Workspace {
  char* base;
  size_t off;
  void* take(size_t bytes) {
    void* p = base + off;
    off += align256(bytes);
    return p;
  }
};

static const int WS_SPINORS64 = 8;   // r,p,t,tmp, b', b^, b-masked, + the source of lqcd_propagator
static const int WS_SPINORS32 = 6;

}  // namespace lqcd

using namespace lqcd;

// Every entry point that takes a geometry runs on the device the geometry was created for (lqcd_geom_desc.device)
// and leaves the caller's current device as it found it.
namespace {
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  explicit DeviceGuard(const lqcd_geom* h) : DeviceGuard(h ? h->desc.device : 0) {}
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
bool good_kappa(const lqcd_dirac* d) { return d->kappa > 0.0 && d->kappa < 1e300; }
}  // namespace

#define REQUIRE(cond, ...)          \
  do {                              \
    if (!(cond)) {                  \
      set_error(__VA_ARGS__);       \
      return LQCD_EINVAL;           \
    }                               \
  } while (0)
#define UNSUPPORTED_ON_SLAB(h, what)                                                                     \
  do {                                                                                                   \
    if ((h)->g.bc == LQCD_BC_SLAB) {                                                                     \
      set_error("%s: not available on a LQCD_BC_SLAB geometry (the time faces would be ignored)", what); \
      return LQCD_EUNSUPPORTED;                                                                          \
    }                                                                                                    \
  } while (0)
#define CUDA_TRY(e, what)                        \
  do {                                           \
    if (!cuda_ok((e), what)) return LQCD_ECUDA;  \
  } while (0)

extern "C" {

const char* lqcd_last_error(void) { return g_err; }
long long lqcd_launch_count(void) { return g_launches.load(); }

lqcd_status lqcd_dw_plan(const lqcd_geom* h, lqcd_prec prec, lqcd_recon recon, int has_clover, int parity, char* buf,
                         int len) {
  REQUIRE(h && buf && len > 0, "lqcd_dw_plan: NULL argument");
  REQUIRE(valid_prec(prec) && valid_recon(recon) && parity >= -1 && parity <= 1, "lqcd_dw_plan: bad precision, link format or parity");
  const int diag = has_clover ? DIAG_PRE : DIAG_ONE;
  const int rc = recon == LQCD_RECON_12 ? 12 : 18;
  if (prec == LQCD_F64) dw_describe<double>(h->g, rc, diag, parity, buf, len);
  else dw_describe<float>(h->g, rc, diag, parity, buf, len);
  return LQCD_OK;
}

lqcd_status lqcd_set_option(const char* key, const char* value) {
  REQUIRE(key && value, "lqcd_set_option: NULL argument");
  if (!strcmp(key, "dw_mode")) {
    REQUIRE(dw_set_mode(value), "lqcd_set_option: dw_mode must be pipe, stream, split or direct");
    return LQCD_OK;
  }
  if (!strcmp(key, "host_slab")) {
    REQUIRE(atoi(value) >= 0, "lqcd_set_option: host_slab must be >= 0");
    lqcd::set_host_slab(atoi(value));
    return LQCD_OK;
  }
  if (!strcmp(key, "pipe_grid")) {
    REQUIRE(dw_set_pipe_grid(atoi(value)), "lqcd_set_option: pipe_grid must be >= 0");
    return LQCD_OK;
  }
  set_error("lqcd_set_option: unknown key '%s'", key);
  return LQCD_EINVAL;
}

lqcd_status lqcd_geom_create(const lqcd_geom_desc* desc, lqcd_geom** out) {
  REQUIRE(desc && out, "lqcd_geom_create: NULL argument");
  *out = nullptr;
  REQUIRE(desc->bc >= LQCD_BC_PERIODIC && desc->bc <= LQCD_BC_SLAB, "lqcd_geom_create: bad bc %d", (int)desc->bc);
  REQUIRE(desc->slab_edges >= 0 && desc->slab_edges <= 5 && (desc->bc == LQCD_BC_SLAB || desc->slab_edges == 0),
          "lqcd_geom_create: bad slab_edges %d", desc->slab_edges);
  for (int i = 0; i < 4; i++)
    REQUIRE(desc->L[i] >= 2 && desc->L[i] % 2 == 0, "lqcd_geom_create: extent L[%d]=%d must be even and >= 2 (R13)", i, desc->L[i]);
  if (desc->bc != LQCD_BC_PERIODIC) REQUIRE(desc->L[3] >= 4, "lqcd_geom_create: open/SF/slab need L[3] >= 4");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    set_error("lqcd_geom_create: no CUDA device (this library has no CPU fallback)");
    return LQCD_ECUDA;
  }
  REQUIRE(desc->device >= 0 && desc->device < ndev, "lqcd_geom_create: bad device %d", desc->device);
  DeviceGuard dg(desc->device);
  lqcd_geom* h = (lqcd_geom*)calloc(1, sizeof(lqcd_geom));
  if (!h) { set_error("out of host memory"); return LQCD_ENOMEM; }
  h->desc = *desc;
  Geom& g = h->g;
  for (int i = 0; i < 4; i++) g.L[i] = desc->L[i];
  g.bc = (int)desc->bc;
  g.edges = desc->bc == LQCD_BC_SLAB ? (desc->slab_edges & 7) : 0;
  g.Vh = (long long)g.L[0] * g.L[1] * g.L[2] * g.L[3] / 2;
  choose_tiling(g);
  h->has_theta = false;
  for (int i = 0; i < 4; i++) {
    double ang = desc->theta[i] / desc->L[i];
    h->th_re[i] = cos(ang);
    h->th_im[i] = sin(ang);
    if (desc->theta[i] != 0.0) h->has_theta = true;
  }
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, desc->device), "cudaGetDeviceProperties");
  h->sm_count = prop.multiProcessorCount;
  h->smem_optin = (int)prop.sharedMemPerBlockOptin;
  g.sm_count = h->sm_count;
  g.smem_optin = h->smem_optin;
  set_reduce_sm_count(h->sm_count);
  {  // neighbour-tile table (a1): 8 neighbours + time origin per tile
    std::vector<int> tab((size_t)g.ntiles * TILE_TAB, 0);
    for (int t = 0; t < g.ntiles; t++) {
      int Tc[4];
      tile_coords(g, t, Tc);
      for (int mu = 0; mu < 4; mu++)
        for (int d = 0; d < 2; d++) {
          int Tn[4] = {Tc[0], Tc[1], Tc[2], Tc[3]};
          Tn[mu] += d ? -1 : +1;
          if (Tn[mu] < 0) Tn[mu] += g.nt[mu];
          if (Tn[mu] >= g.nt[mu]) Tn[mu] -= g.nt[mu];
          tab[(size_t)t * TILE_TAB + 2 * mu + d] = tile_linear(g, Tn[0], Tn[1], Tn[2], Tn[3]);
        }
      tab[(size_t)t * TILE_TAB + 8] = Tc[3] * g.b[3];
      for (int i = 0; i < 3; i++) tab[(size_t)t * TILE_TAB + 9 + i] = Tc[i] * g.b[i];   // spatial origin of the tile
    }
    int* dtab = nullptr;
    if (!cuda_ok(cudaMalloc(&dtab, tab.size() * sizeof(int)), "cudaMalloc(tile table)")) { free(h); return LQCD_ENOMEM; }
    if (!cuda_ok(cudaMemcpy(dtab, tab.data(), tab.size() * sizeof(int), cudaMemcpyHostToDevice), "cudaMemcpy(tile table)")) {
      cudaFree(dtab); free(h); return LQCD_ECUDA;
    }
    g.tile_tab = dtab;
    unsigned int* sched = nullptr;
    if (!cuda_ok(cudaMalloc(&sched, SCHED_SLOTS * 2 * sizeof(unsigned int)), "cudaMalloc(scheduler)") ||
        !cuda_ok(cudaMemset(sched, 0, SCHED_SLOTS * 2 * sizeof(unsigned int)), "cudaMemset(scheduler)")) {
      cudaFree(sched); cudaFree(dtab); free(h); return LQCD_ECUDA;
    }
    g.sched = sched;
  }
  *out = h;
  return LQCD_OK;
}

lqcd_status lqcd_geom_destroy(lqcd_geom* g) {
  if (g) {
    DeviceGuard dg(g);
    if (g->g.tile_tab) cudaFree((void*)g->g.tile_tab);
    if (g->g.sched) cudaFree((void*)g->g.sched);
    free(g);
  }
  return LQCD_OK;
}

lqcd_status lqcd_geom_info(const lqcd_geom* h, int tile[4], int ntiles[4], int chunk[2]) {
  REQUIRE(h, "lqcd_geom_info: NULL geometry");
  for (int i = 0; i < 4; i++) {
    if (tile) tile[i] = h->g.b[i];
    if (ntiles) ntiles[i] = h->g.nt[i];
  }
  if (chunk) { chunk[0] = h->g.c1; chunk[1] = h->g.c2; }
  return LQCD_OK;
}

size_t lqcd_field_bytes(const lqcd_geom* h, lqcd_field_kind kind, lqcd_prec prec, lqcd_recon recon) {
  if (!h) return 0;
  const Geom& g = h->g;
  size_t sites = (size_t)2 * g.Vh;
  size_t eb = elem_bytes(prec);
  switch (kind) {
    case LQCD_FIELD_GAUGE: return sites * 4 * (recon == LQCD_RECON_12 ? 6 : 9) * eb;
    case LQCD_FIELD_SPINOR: return sites * 12 * eb;
    case LQCD_FIELD_CLOVER: return sites * 36 * eb;
    case LQCD_FIELD_FACE: return (size_t)g.L[0] * g.L[1] * g.L[2] * 6 * eb;
    case LQCD_FIELD_WORKSPACE: {
      size_t sp64 = align256(sites * 12 * sizeof(double2)), sp32 = align256(sites * 12 * sizeof(float2));
      return WS_SPINORS64 * sp64 + WS_SPINORS32 * sp32 + 2 * align256(partial_len(g) * sizeof(double)) + 4096;
    }
  }
  return 0;
}

#define DISPATCH_PREC(prec, call_d, call_f) ((prec) == LQCD_F64 ? (call_d) : (call_f))

lqcd_status lqcd_gauge_import(const lqcd_geom* h, const void* canon, void* U, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && canon && U && canon != U, "lqcd_gauge_import: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_gauge_import: bad precision / recon");
  CUDA_TRY(DISPATCH_PREC(prec, gauge_import<double>(h->g, canon, U, recon, as_stream(stream)),
                         gauge_import<float>(h->g, canon, U, recon, as_stream(stream))), "gauge_import");
  return LQCD_OK;
}
lqcd_status lqcd_gauge_export(const lqcd_geom* h, const void* U, void* canon, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && canon && U && canon != U, "lqcd_gauge_export: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_gauge_export: bad precision / recon");
  CUDA_TRY(DISPATCH_PREC(prec, gauge_export<double>(h->g, U, canon, recon, as_stream(stream)),
                         gauge_export<float>(h->g, U, canon, recon, as_stream(stream))), "gauge_export");
  return LQCD_OK;
}
lqcd_status lqcd_spinor_import(const lqcd_geom* h, const void* canon, void* psi, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && psi && canon != psi, "lqcd_spinor_import: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_spinor_import: bad precision");
  CUDA_TRY(DISPATCH_PREC(prec, spinor_import<double>(h->g, canon, psi, as_stream(stream)),
                         spinor_import<float>(h->g, canon, psi, as_stream(stream))), "spinor_import");
  return LQCD_OK;
}
lqcd_status lqcd_spinor_export(const lqcd_geom* h, const void* psi, void* canon, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && psi && canon != psi, "lqcd_spinor_export: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_spinor_export: bad precision");
  CUDA_TRY(DISPATCH_PREC(prec, spinor_export<double>(h->g, psi, canon, as_stream(stream)),
                         spinor_export<float>(h->g, psi, canon, as_stream(stream))), "spinor_export");
  return LQCD_OK;
}
lqcd_status lqcd_clover_export(const lqcd_geom* h, const void* clover, void* canon, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && clover && canon != clover, "lqcd_clover_export: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_clover_export: bad precision");
  CUDA_TRY(DISPATCH_PREC(prec, clover_export<double>(h->g, clover, canon, as_stream(stream)),
                         clover_export<float>(h->g, clover, canon, as_stream(stream))), "clover_export");
  return LQCD_OK;
}
lqcd_status lqcd_field_to_f32(const lqcd_geom* h, lqcd_field_kind kind, lqcd_recon recon, const void* src64, void* dst32, void* stream) {
  REQUIRE(h && src64 && dst32 && src64 != dst32, "lqcd_field_to_f32: NULL or aliased argument");
  DeviceGuard dg(h);
  REQUIRE(kind == LQCD_FIELD_GAUGE || kind == LQCD_FIELD_SPINOR || kind == LQCD_FIELD_CLOVER, "lqcd_field_to_f32: bad kind");
  size_t n = lqcd_field_bytes(h, kind, LQCD_F64, recon) / sizeof(double2);
  CUDA_TRY(to_f32(src64, dst32, n, as_stream(stream)), "to_f32");
  return LQCD_OK;
}

lqcd_status lqcd_clover_build(const lqcd_geom* h, const lqcd_dirac* d, const void* U64, lqcd_recon recon, void* clover,
                              void* clover_inv, lqcd_prec out_prec, void* stream) {
  REQUIRE(h && d && U64 && clover, "lqcd_clover_build: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_clover_build: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(valid_prec(out_prec) && valid_recon(recon), "lqcd_clover_build: bad precision / recon");
  REQUIRE(clover != U64 && clover_inv != U64 && clover != clover_inv, "lqcd_clover_build: aliased buffers");
  UNSUPPORTED_ON_SLAB(h, "lqcd_clover_build (use lqcd_clover_build_slab)");
  CloverParm cp;
  cp.kappa = d->kappa; cp.csw = d->csw; cp.ct = d->ct;
  for (int i = 0; i < 3; i++) cp.phiT[i] = h->desc.phiT[i];
  CUDA_TRY(clover_build(h->g, cp, U64, (int)recon, clover, clover_inv, (int)out_prec, as_stream(stream)), "clover_build");
  return LQCD_OK;
}

lqcd_status lqcd_clover_build_slab(const lqcd_geom* h, const lqcd_dirac* d, const void* U64, lqcd_recon recon,
                                   const void* halo_lo, const void* halo_hi, void* clover, void* clover_inv,
                                   lqcd_prec out_prec, void* stream) {
  REQUIRE(h && d && U64 && clover, "lqcd_clover_build_slab: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_clover_build_slab: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(h->g.bc == LQCD_BC_SLAB, "lqcd_clover_build_slab: the geometry is not a slab (bc != LQCD_BC_SLAB)");
  REQUIRE((halo_lo || (h->g.edges & LQCD_SLAB_OPEN_LO)) && (halo_hi || (h->g.edges & (LQCD_SLAB_OPEN_HI | LQCD_SLAB_SF_HI))),
          "lqcd_clover_build_slab: a gauge halo is required on every face that is not an open boundary");
  REQUIRE(valid_prec(out_prec) && valid_recon(recon), "lqcd_clover_build_slab: bad precision / recon");
  REQUIRE(clover != U64 && clover_inv != U64 && clover != clover_inv, "lqcd_clover_build_slab: aliased buffers");
  CloverParm cp;
  cp.kappa = d->kappa; cp.csw = d->csw; cp.ct = d->ct;
  for (int i = 0; i < 3; i++) cp.phiT[i] = h->desc.phiT[i];
  CUDA_TRY(clover_build(h->g, cp, U64, (int)recon, clover, clover_inv, (int)out_prec, as_stream(stream), halo_lo, halo_hi),
           "clover_build (slab)");
  return LQCD_OK;
}

lqcd_status lqcd_dw_slab_pack(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* in, void* send_lo,
                              void* send_hi, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && U && in && send_lo && send_hi, "lqcd_dw_slab_pack: NULL argument");
  DeviceGuard dg(h);
  REQUIRE(h->g.bc == LQCD_BC_SLAB, "lqcd_dw_slab_pack: the geometry is not a slab (bc != LQCD_BC_SLAB)");
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_slab_pack: bad precision / recon");
  REQUIRE(send_lo != send_hi, "lqcd_dw_slab_pack: aliased face buffers");
  CUDA_TRY(DISPATCH_PREC(prec, slab_pack<double>(h, dagger != 0, U, (int)recon, in, send_lo, send_hi, as_stream(stream)),
                         slab_pack<float>(h, dagger != 0, U, (int)recon, in, send_lo, send_hi, as_stream(stream))),
           "slab_pack kernel");
  return LQCD_OK;
}

lqcd_status lqcd_dw_slab_faces(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* recv_lo,
                               const void* recv_hi, void* out, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && U && recv_lo && recv_hi && out, "lqcd_dw_slab_faces: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_dw_slab_faces: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(h->g.bc == LQCD_BC_SLAB, "lqcd_dw_slab_faces: the geometry is not a slab (bc != LQCD_BC_SLAB)");
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_slab_faces: bad precision / recon");
  CUDA_TRY(DISPATCH_PREC(prec, slab_faces<double>(h, d->kappa, dagger != 0, U, (int)recon, recv_lo, recv_hi, out, as_stream(stream)),
                         slab_faces<float>(h, d->kappa, dagger != 0, U, (int)recon, recv_lo, recv_hi, out, as_stream(stream))),
           "slab_faces kernel");
  return LQCD_OK;
}

}  // extern "C"
template <typename T>
static cudaError_t dw_apply_t(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                              void* out, bool dagger, int recon, cudaStream_t s) {
  Op<T> M;
  M.geom = h; M.U = U; M.A = clover; M.Ainv = nullptr; M.tmp = nullptr; M.kappa = d->kappa; M.mu = d->mu; M.recon = recon; M.eo = false;
  return M.apply(in, out, dagger, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s);
}

template <typename T>
static cudaError_t dw_multi_t(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                              void* out, int nrhs, bool dagger, int recon, cudaStream_t s) {
  Op<T> M;
  M.geom = h; M.U = U; M.A = clover; M.Ainv = nullptr; M.tmp = nullptr; M.kappa = d->kappa; M.mu = d->mu; M.recon = recon; M.eo = false;
  return M.apply_multi(in, out, nrhs, dagger, s);
}

extern "C" {
lqcd_status lqcd_dw_apply_multi(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                                void* out, int nrhs, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && U && in && out, "lqcd_dw_apply_multi: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_dw_apply_multi: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_apply_multi: bad precision / recon");
  REQUIRE(nrhs >= 1 && nrhs <= 64, "lqcd_dw_apply_multi: nrhs must be in 1..64");
  const size_t fb = lqcd_field_bytes(h, LQCD_FIELD_SPINOR, prec, recon);
  const char *ib = (const char*)in, *ob = (const char*)out;
  REQUIRE(ob + nrhs * fb <= ib || ib + nrhs * fb <= ob, "lqcd_dw_apply_multi: input and output arrays overlap");
  REQUIRE(out != U && out != clover, "lqcd_dw_apply_multi: output aliases an input");
  CUDA_TRY(DISPATCH_PREC(prec, dw_multi_t<double>(h, d, U, clover, in, out, nrhs, dagger != 0, (int)recon, as_stream(stream)),
                         dw_multi_t<float>(h, d, U, clover, in, out, nrhs, dagger != 0, (int)recon, as_stream(stream))),
           "dw kernel (multi)");
  return LQCD_OK;
}
static lqcd_status dw_common(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                             void* out, lqcd_prec prec, lqcd_recon recon, void* stream, bool dagger) {
  REQUIRE(h && d && U && in && out, "lqcd_dw_apply: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_dw_apply: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_apply: bad precision / recon");
  REQUIRE(out != in && out != U && out != clover, "lqcd_dw_apply: output aliases an input (PAPER.md:121: separate pso/psi)");
  CUDA_TRY(DISPATCH_PREC(prec, dw_apply_t<double>(h, d, U, clover, in, out, dagger, (int)recon, as_stream(stream)),
                         dw_apply_t<float>(h, d, U, clover, in, out, dagger, (int)recon, as_stream(stream))), "dw kernel");
  return LQCD_OK;
}
lqcd_status lqcd_dw_apply(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                          void* out, lqcd_prec prec, lqcd_recon recon, void* stream) {
  return dw_common(h, d, U, clover, in, out, prec, recon, stream, false);
}
lqcd_status lqcd_dwdag_apply(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                             void* out, lqcd_prec prec, lqcd_recon recon, void* stream) {
  return dw_common(h, d, U, clover, in, out, prec, recon, stream, true);
}

}  // extern "C"
template <typename T>
static cudaError_t dw_eo_t(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* A, const void* Ainv,
                           const void* in, void* out, void* tmp, bool dagger, int recon, cudaStream_t s) {
  Op<T> M;
  M.geom = h; M.U = U; M.A = A; M.Ainv = Ainv; M.tmp = tmp; M.kappa = d->kappa; M.recon = recon; M.eo = true;
  return M.apply(in, out, dagger, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s);
}
extern "C" {
lqcd_status lqcd_dw_eo_apply(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* clover_inv,
                             const void* in_e, void* out_e, void* tmp, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && U && clover && clover_inv && in_e && out_e && tmp, "lqcd_dw_eo_apply: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_dw_eo_apply: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_eo_apply: bad precision / recon");
  REQUIRE(out_e != in_e && tmp != in_e && tmp != out_e, "lqcd_dw_eo_apply: aliased buffers");
  REQUIRE(d->mu == 0.0, "lqcd_dw_eo_apply: the even-odd operator does not support a twisted mass (mu != 0)");
  UNSUPPORTED_ON_SLAB(h, "lqcd_dw_eo_apply");
  CUDA_TRY(DISPATCH_PREC(prec, dw_eo_t<double>(h, d, U, clover, clover_inv, in_e, out_e, tmp, dagger != 0, (int)recon, as_stream(stream)),
                         dw_eo_t<float>(h, d, U, clover, clover_inv, in_e, out_e, tmp, dagger != 0, (int)recon, as_stream(stream))),
           "dw_eo kernel");
  return LQCD_OK;
}

lqcd_status lqcd_point_source(const lqcd_geom* h, const int y[4], int spin, int colour, void* b, lqcd_prec prec, void* stream) {
  REQUIRE(h && y && b, "lqcd_point_source: NULL argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_point_source: bad precision");
  REQUIRE(spin >= 0 && spin < 4 && colour >= 0 && colour < 3, "lqcd_point_source: bad spin/colour");
  for (int i = 0; i < 4; i++) REQUIRE(y[i] >= 0 && y[i] < h->g.L[i], "lqcd_point_source: position outside the lattice");
  CUDA_TRY(DISPATCH_PREC(prec, point_source<double>(h->g, y, spin, colour, b, as_stream(stream)),
                         point_source<float>(h->g, y, spin, colour, b, as_stream(stream))), "point_source");
  return LQCD_OK;
}

lqcd_status lqcd_spinor_norm2(const lqcd_geom* h, const void* v, int half, lqcd_prec prec, void* workspace, double* result_host, void* stream) {
  REQUIRE(h && v && workspace && result_host, "lqcd_spinor_norm2: NULL argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_spinor_norm2: bad precision");
  size_t n = spinor_complex(h->g) / (half ? 2 : 1);
  double* partial = (double*)workspace;
  double* scratch = partial + partial_len(h->g) - 8;
  CUDA_TRY(DISPATCH_PREC(prec, device_norm2<double>(v, n, partial, scratch, result_host, as_stream(stream)),
                         device_norm2<float>(v, n, partial, scratch, result_host, as_stream(stream))), "norm2");
  return LQCD_OK;
}
lqcd_status lqcd_correlator_ps(const lqcd_geom* h, const void* columns, int ncol, lqcd_prec prec, void* workspace,
                               double* C_host, void* stream) {
  REQUIRE(h && columns && workspace && C_host, "lqcd_correlator_ps: NULL argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec) && ncol >= 1 && ncol <= 4096, "lqcd_correlator_ps: bad precision or column count");
  const Geom& g = h->g;
  double* partial = (double*)workspace;   // the workspace is several spinor fields large: ntiles*b3 + L4 doubles fit
  double* C_dev = partial + (size_t)g.ntiles * g.b[3];
  cudaStream_t s = as_stream(stream);
  CUDA_TRY(DISPATCH_PREC(prec, correlator_ps<double>(g, columns, ncol, partial, C_dev, s),
                         correlator_ps<float>(g, columns, ncol, partial, C_dev, s)), "correlator kernel");
  CUDA_TRY(cudaMemcpyAsync(C_host, C_dev, (size_t)g.L[3] * sizeof(double), cudaMemcpyDeviceToHost, s), "memcpy");
  CUDA_TRY(cudaStreamSynchronize(s), "sync");
  return LQCD_OK;
}
lqcd_status lqcd_spinor_dot(const lqcd_geom* h, const void* u, const void* v, int half, lqcd_prec prec, void* workspace, double* result_host, void* stream) {
  REQUIRE(h && u && v && workspace && result_host, "lqcd_spinor_dot: NULL argument");
  DeviceGuard dg(h);
  REQUIRE(valid_prec(prec), "lqcd_spinor_dot: bad precision");
  size_t n = spinor_complex(h->g) / (half ? 2 : 1);
  double* partial = (double*)workspace;
  double* scratch = partial + partial_len(h->g) - 8;
  cudaStream_t s = as_stream(stream);
  CUDA_TRY(DISPATCH_PREC(prec, dot_partial<double>(u, v, n, partial, s), dot_partial<float>(u, v, n, partial, s)), "dot");
  CUDA_TRY(final_sum(partial, reduce_blocks(n), 2, scratch, s), "final_sum");
  CUDA_TRY(cudaMemcpyAsync(result_host, scratch, 2 * sizeof(double), cudaMemcpyDeviceToHost, s), "memcpy");
  CUDA_TRY(cudaStreamSynchronize(s), "sync");
  return LQCD_OK;
}

}  // extern "C"
// ---------------------------------------------------------------------------------------------------------
// solver
// ---------------------------------------------------------------------------------------------------------
namespace {

struct SolveCtx {
  const lqcd_geom* h;
  const lqcd_dirac* d;
  const lqcd_cg_fields* f;
  const lqcd_cg_parm* parm;
  int recon;
  cudaStream_t s;
  // workspace pieces
  void* v64[WS_SPINORS64];
  void* v32[WS_SPINORS32];
  double* partial;
  double* scratch;     // 8 doubles on the device
  CgState* state;
  unsigned int* sched = nullptr;   // SCHED_POOL_PAIRS zeroed counter pairs (CgVectors::sched_pool)
};

template <typename T>
Op<T> make_op(const SolveCtx& c, void* tmp) {
  Op<T> M;
  M.geom = c.h;
  const bool f64 = sizeof(T) == 8;
  M.U = f64 ? c.f->U64 : c.f->U32;
  M.A = f64 ? c.f->clover64 : c.f->clover32;
  M.Ainv = f64 ? c.f->clover_inv64 : c.f->clover_inv32;
  M.tmp = tmp;
  M.kappa = c.d->kappa;
  M.mu = c.d->mu;
  M.recon = c.recon;
  M.eo = c.parm->eo != 0;
  return M;
}

#define CKS(e, what) do { if (!cuda_ok((e), what)) return LQCD_ECUDA; } while (0)

// Solve M^+ M x = bp in fp64, plain or by defect correction with an fp32 inner CG.
// Uses v64[0..2] (r,p,t), v64[3] (tmp for eo) and the fp32 vectors.  Returns iterations in *iters, outer count in *outer.
lqcd_status solve_normal(const SolveCtx& c, const void* bp, void* x, int* iters, int* outer, double* rho0_out) {
  Op<double> M = make_op<double>(c, c.v64[3]);
  const size_t n = M.ncomplex();
  CgVectors v;
  v.r = c.v64[0]; v.p = c.v64[1]; v.t = c.v64[2]; v.partial = c.partial; v.state = c.state; v.sched_pool = c.sched;
  CgState hs;
  const int check = c.parm->check_every > 0 ? c.parm->check_every : 16;
  *outer = 0;
  if (!c.parm->mixed) {
    CKS(cg_normal<double>(M, bp, x, v, c.parm->tol, c.parm->maxiter, check, &hs, c.s), "cg_normal");
    *iters = hs.iters;
    *rho0_out = hs.rho0;
    if (hs.breakdown) { set_error("lqcd_cg_solve: breakdown (NaN or <p,M^+M p> <= 0) at iteration %d", hs.iters); return LQCD_EBREAKDOWN; }
    if (!hs.done) { set_error("lqcd_cg_solve: not converged after %d iterations", hs.iters); return LQCD_ENOTCONV; }
    return LQCD_OK;
  }
  // mixed precision: r = bp - M^+M x (fp64); e = CG32(r) to inner_tol; x += e
  Op<float> M32 = make_op<float>(c, c.v32[4]);
  CgVectors w;
  w.r = c.v32[1]; w.p = c.v32[2]; w.t = c.v32[3]; w.partial = c.partial; w.state = c.state; w.sched_pool = c.sched;
  void* r64 = c.v64[0];
  void* t64 = c.v64[1];
  void* q64 = c.v64[2];
  double rho0 = 0, rho = 0;
  CKS(cudaMemsetAsync(x, 0, n * sizeof(double2), c.s), "memset");
  CKS(cudaMemcpyAsync(r64, bp, n * sizeof(double2), cudaMemcpyDeviceToDevice, c.s), "copy");
  CKS(device_norm2<double>(r64, n, c.partial, c.scratch, &rho0, c.s), "norm2");
  *rho0_out = rho0;
  rho = rho0;
  int total = 0;
  const double inner_tol = c.parm->inner_tol > 0 ? c.parm->inner_tol : 1e-4;
  for (;;) {
    if (rho0 == 0.0 || rho <= c.parm->tol * c.parm->tol * rho0) break;
    if (!(rho == rho)) { *iters = total; set_error("lqcd_cg_solve: NaN residual in mixed solve"); return LQCD_EBREAKDOWN; }
    if (total >= c.parm->maxiter) { *iters = total; set_error("lqcd_cg_solve: not converged after %d inner iterations", total); return LQCD_ENOTCONV; }
    CKS(to_f32(r64, c.v32[0], n, c.s), "to_f32");
    // do not ask the inner solve for more than the outer one still needs
    double need = c.parm->tol * sqrt(rho0 / rho) * 0.5;
    double itol = inner_tol > need ? inner_tol : need;
    CKS(cg_normal<float>(M32, c.v32[0], c.v32[5], w, itol, c.parm->maxiter - total, check, &hs, c.s), "cg_normal32");
    total += hs.iters;
    *outer += 1;
    if (getenv("LQCD_CG_VERBOSE"))
      fprintf(stderr, "lqcd_cg_solve mixed: outer %d: |r|/|b'| = %.3e before, inner tol %.1e, inner iterations %d (inner recursive |r|^2 ratio %.3e)\n",
              *outer, sqrt(rho / rho0), itol, hs.iters, hs.rho0 > 0 ? hs.rho / hs.rho0 : 0.0);
    if (hs.breakdown) { *iters = total; set_error("lqcd_cg_solve: breakdown in the fp32 inner solve"); return LQCD_EBREAKDOWN; }
    CKS(add_f32_to_f64(c.v32[5], x, n, c.s), "x += e");
    CKS(M.apply(x, t64, false, EPI_STORE, nullptr, nullptr, nullptr, nullptr, c.s), "M x");
    CKS(M.apply(t64, q64, true, EPI_STORE, nullptr, nullptr, nullptr, nullptr, c.s), "M^+ M x");
    CKS(xmy<double>(bp, q64, r64, n, c.s), "r = bp - q");
    CKS(device_norm2<double>(r64, n, c.partial, c.scratch, &rho, c.s), "norm2");
  }
  *iters = total;
  return LQCD_OK;
}

}  // namespace

extern "C" {
lqcd_status lqcd_cg_solve(const lqcd_geom* h, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b, void* x,
                          void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && f && b && x && workspace && parm && info, "lqcd_cg_solve: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_cg_solve: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(valid_recon(recon), "lqcd_cg_solve: bad recon");
  REQUIRE(f->U64, "lqcd_cg_solve: U64 is required");
  REQUIRE(x != b, "lqcd_cg_solve: x aliases b");
  UNSUPPORTED_ON_SLAB(h, "lqcd_cg_solve");
  REQUIRE(parm->tol > 0 && parm->maxiter >= 0, "lqcd_cg_solve: bad tol / maxiter");
  if (parm->eo) REQUIRE(f->clover64 && f->clover_inv64, "lqcd_cg_solve: eo needs clover64 and clover_inv64");
  if (parm->eo) REQUIRE(d->mu == 0.0, "lqcd_cg_solve: the even-odd solver does not support a twisted mass (mu != 0)");
  if (parm->mixed) {
    REQUIRE(f->U32, "lqcd_cg_solve: mixed needs U32");
    REQUIRE((f->clover64 == nullptr) == (f->clover32 == nullptr), "lqcd_cg_solve: mixed needs clover32 iff clover64");
    if (parm->eo) REQUIRE(f->clover_inv32, "lqcd_cg_solve: mixed eo needs clover_inv32");
  }
  memset(info, 0, sizeof(*info));
  auto t0 = std::chrono::steady_clock::now();
  const Geom& g = h->g;
  SolveCtx c;
  c.h = h; c.d = d; c.f = f; c.parm = parm; c.recon = (int)recon; c.s = as_stream(stream);
  Workspace ws{(char*)workspace, 0};
  const size_t sites = (size_t)2 * g.Vh;
  for (int i = 0; i < WS_SPINORS64; i++) c.v64[i] = ws.take(sites * 12 * sizeof(double2));
  for (int i = 0; i < WS_SPINORS32; i++) c.v32[i] = ws.take(sites * 12 * sizeof(float2));
  c.partial = (double*)ws.take(partial_len(g) * sizeof(double));
  c.scratch = (double*)ws.take(64);
  c.state = (CgState*)ws.take(sizeof(CgState));
  c.sched = (unsigned int*)ws.take((size_t)SCHED_POOL_PAIRS * 2 * sizeof(unsigned int));
  CKS(cudaMemsetAsync(c.sched, 0, (size_t)SCHED_POOL_PAIRS * 2 * sizeof(unsigned int), as_stream(stream)), "memset");
  const size_t nfull = spinor_complex(g);
  cudaStream_t s = c.s;
  lqcd_status st = LQCD_OK;
  double rho0 = 0;
  int iters = 0, outer = 0;

  if (!parm->eo) {
    Op<double> M = make_op<double>(c, nullptr);
    void* bp = c.v64[4];
    if (g.bc != LQCD_BC_PERIODIC) {
      // D7: the solve lives on the interior; components of b on frozen slices are ignored (as in the even-odd branch),
      // so that |b| and b - Dx below do not count them
      void* bm = c.v64[6];
      CKS(cudaMemcpyAsync(bm, b, nfull * sizeof(double2), cudaMemcpyDeviceToDevice, s), "copy b");
      CKS(mask_frozen<double>(g, bm, s), "mask");
      b = bm;
    }
    CKS(M.apply(b, bp, true, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D^+ b");
    st = solve_normal(c, bp, x, &iters, &outer, &rho0);
    if (st != LQCD_OK && st != LQCD_ENOTCONV) { info->iters = iters; info->outer = outer; return st; }
    // true residuals with fresh operator applications (R11)
    void* t = c.v64[0];
    void* q = c.v64[1];
    double nb = 0, nr = 0, nq = 0;
    CKS(M.apply(x, t, false, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D x");
    CKS(xmy<double>(b, t, t, nfull, s), "b - Dx");
    CKS(device_norm2<double>(b, nfull, c.partial, c.scratch, &nb, s), "norm2");
    CKS(device_norm2<double>(t, nfull, c.partial, c.scratch, &nr, s), "norm2");
    CKS(M.apply(t, q, true, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D^+ (b - Dx)");
    CKS(device_norm2<double>(q, nfull, c.partial, c.scratch, &nq, s), "norm2");
    info->rel_resid_true = nb > 0 ? sqrt(nr / nb) : 0.0;
    info->rel_resid_normal = rho0 > 0 ? sqrt(nq / rho0) : 0.0;
  } else {
    // D8: b^_e = b_e + kappa H_eo A_oo^{-1} b_o ; solve D^ x_e = b^_e ; x_o = A_oo^{-1} (b_o + kappa H_oe x_e)
    Op<double> M = make_op<double>(c, c.v64[3]);
    void* tmp = c.v64[3];   // full field scratch (odd half used)
    void* bh = c.v64[4];    // b^_e   (even half)
    void* bp = c.v64[5];    // D^^+ b^_e
    void* bm = c.v64[6];    // b with the frozen slices zeroed
    CKS(cudaMemcpyAsync(bm, b, nfull * sizeof(double2), cudaMemcpyDeviceToDevice, s), "copy b");
    CKS(mask_frozen<double>(g, bm, s), "mask");
    CKS(launch_diag<double>(g, f->clover_inv64, bm, tmp, 1, s), "A_oo^-1 b_o");
    CKS(M.hop_xpay(tmp, bm, bh, -d->kappa, 0, s), "b_e + kappa H_eo .");
    CKS(M.apply(bh, bp, true, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D^^+ b^");
    st = solve_normal(c, bp, x, &iters, &outer, &rho0);   // x even half
    if (st != LQCD_OK && st != LQCD_ENOTCONV) { info->iters = iters; info->outer = outer; return st; }
    // normal-equation residual of the preconditioned system
    {
      void* t = c.v64[0];
      void* q = c.v64[1];
      double nq = 0;
      const size_t nh = nfull / 2;
      CKS(M.apply(x, t, false, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D^ x");
      CKS(xmy<double>(bh, t, t, nh, s), "b^ - D^ x");
      CKS(M.apply(t, q, true, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D^^+ .");
      CKS(device_norm2<double>(q, nh, c.partial, c.scratch, &nq, s), "norm2");
      info->rel_resid_normal = rho0 > 0 ? sqrt(nq / rho0) : 0.0;
    }
    // odd part: tmp_o = b_o + kappa H_oe x_e ; x_o = A_oo^{-1} tmp_o   (x is a full field: even half solved above)
    CKS(M.hop_xpay(x, bm, tmp, -d->kappa, 1, s), "b_o + kappa H_oe x_e");
    CKS(launch_diag<double>(g, f->clover_inv64, tmp, x, 1, s), "A_oo^-1 .");
    // true residual of the full system
    {
      Op<double> Mf = make_op<double>(c, nullptr);
      Mf.eo = false;
      void* t = c.v64[0];
      double nb = 0, nr = 0;
      CKS(Mf.apply(x, t, false, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "D x");
      CKS(xmy<double>(bm, t, t, nfull, s), "b - Dx");
      CKS(device_norm2<double>(bm, nfull, c.partial, c.scratch, &nb, s), "norm2");
      CKS(device_norm2<double>(t, nfull, c.partial, c.scratch, &nr, s), "norm2");
      info->rel_resid_true = nb > 0 ? sqrt(nr / nb) : 0.0;
    }
  }
  CKS(cudaStreamSynchronize(s), "sync");
  info->iters = iters;
  info->outer = outer;
  info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  return st;
}

}  // extern "C"

// ---- NEXT-3: CG over the time slabs of a decomposed lattice -------------------------------------------------------
namespace {
#define LSS(e) do { lqcd_status _st = (e); if (_st != LQCD_OK) return _st; } while (0)

template <typename T>
struct SlabSolve {
  const lqcd_geom* h;
  const lqcd_dirac* d;
  const void* U;
  const void* A;
  int recon;
  const lqcd_slab_comm* comm;
  double* partial;
  cudaStream_t s;

  size_t face_bytes() const { return (size_t)h->g.L[0] * h->g.L[1] * h->g.L[2] * 6 * 2 * sizeof(T); }
  lqcd_status cb(int rc, const char* what) const {
    if (rc != 0) { set_error("lqcd_cg_solve_slab: callback %s failed (%d)", what, rc); return LQCD_ECUDA; }
    return LQCD_OK;
  }
  // out = D in (D^+ in) on this rank's slab, faces included
  lqcd_status apply(const void* in, void* out, bool dagger) const {
    CKS(slab_pack<T>(h, dagger, U, recon, in, comm->send_lo, comm->send_hi, s), "slab_pack");
    LSS(cb(comm->exchange_start(comm->ctx, face_bytes()), "exchange_start"));
    Op<T> M;
    M.geom = h; M.U = U; M.A = A; M.Ainv = nullptr; M.tmp = nullptr; M.kappa = d->kappa; M.mu = d->mu; M.recon = recon; M.eo = false;
    CKS(M.apply(in, out, dagger, EPI_STORE, nullptr, nullptr, nullptr, nullptr, s), "slab stencil");
    LSS(cb(comm->exchange_wait(comm->ctx), "exchange_wait"));
    CKS(slab_faces<T>(h, d->kappa, dagger, U, recon, comm->recv_lo, comm->recv_hi, out, s), "slab_faces");
    return LQCD_OK;
  }
  // scalars[0] = sum over ranks of the `nblocks` partial sums in `partial`
  lqcd_status reduce(int nblocks) const {
    CKS(final_sum(partial, nblocks, 1, comm->scalars, s), "final_sum");
    return cb(comm->allreduce_sum(comm->ctx, 1), "allreduce_sum");
  }
  lqcd_status norm2(const void* v, size_t n, double* host) const {
    CKS(norm2_partial<T>(v, n, partial, s), "norm2");
    LSS(reduce(reduce_blocks(n)));
    if (host) {
      CKS(cudaMemcpyAsync(host, comm->scalars, sizeof(double), cudaMemcpyDeviceToHost, s), "copy scalar");
      CKS(cudaStreamSynchronize(s), "sync");
    }
    return LQCD_OK;
  }
  // CG on D^+D x = bp from x = 0 (the algorithm of cg_normal; unfused residual update, all-reduced scalars).
  // Every rank sees the same all-reduced scalars, hence the same state: the ranks stay in lockstep.
  lqcd_status cg(const void* bp, void* x, void* r, void* p, void* t, void* q, CgState* state, double tol, int maxiter,
                 int check, CgState* hs) const {
    typedef typename vec2<T>::type T2;
    const size_t n = spinor_complex(h->g);
    const size_t bytes = n * sizeof(T2);
    CKS(cudaMemsetAsync(x, 0, bytes, s), "memset");
    CKS(cudaMemcpyAsync(r, bp, bytes, cudaMemcpyDeviceToDevice, s), "copy");
    CKS(cudaMemcpyAsync(p, bp, bytes, cudaMemcpyDeviceToDevice, s), "copy");
    LSS(norm2(r, n, nullptr));
    CKS(cg_init_state(state, comm->scalars, 1, tol, s), "cg_init_state");
    int launched = 0;
    for (;;) {
      CKS(cudaMemcpyAsync(hs, state, sizeof(CgState), cudaMemcpyDeviceToHost, s), "copy state");
      CKS(cudaStreamSynchronize(s), "sync");
      if (hs->done || launched >= maxiter) break;
      int batch = check;
      if (launched + batch > maxiter) batch = maxiter - launched;
      for (int it = 0; it < batch; it++) {
        LSS(apply(p, t, false));
        CKS(norm2_partial<T>(t, n, partial, s), "norm2");
        LSS(reduce(reduce_blocks(n)));
        CKS(cg_reduce_alpha(state, comm->scalars, 1, s), "alpha");
        LSS(apply(t, q, true));
        CKS(cg_raxpy_norm<T>(state, q, r, n, partial, s), "r -= alpha q");
        LSS(reduce(reduce_blocks(n)));
        CKS(cg_reduce_beta(state, comm->scalars, 1, s), "beta");
        CKS(cg_update_xp<T>(state, x, p, r, n, s), "update");
      }
      launched += batch;
    }
    return LQCD_OK;
  }
};
}  // namespace

extern "C" lqcd_status lqcd_cg_solve_slab(const lqcd_geom* h, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b,
                                          void* x, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info,
                                          const lqcd_slab_comm* comm, lqcd_recon recon, void* stream) {
  REQUIRE(h && d && f && b && x && workspace && parm && info && comm, "lqcd_cg_solve_slab: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_cg_solve_slab: kappa must be positive and finite (got %g)", d->kappa);
  DeviceGuard dg(h);
  REQUIRE(h->g.bc == LQCD_BC_SLAB, "lqcd_cg_solve_slab: the geometry is not a slab (bc != LQCD_BC_SLAB)");
  REQUIRE(valid_recon(recon), "lqcd_cg_solve_slab: bad recon");
  REQUIRE(f->U64, "lqcd_cg_solve_slab: U64 is required");
  REQUIRE(x != b, "lqcd_cg_solve_slab: x aliases b");
  REQUIRE(parm->tol > 0 && parm->maxiter >= 0, "lqcd_cg_solve_slab: bad tol / maxiter");
  REQUIRE(!parm->eo, "lqcd_cg_solve_slab: the even-odd operator is not available on slabs (eo must be 0)");
  if (parm->mixed) {
    REQUIRE(f->U32, "lqcd_cg_solve_slab: mixed needs U32");
    REQUIRE((f->clover64 == nullptr) == (f->clover32 == nullptr), "lqcd_cg_solve_slab: mixed needs clover32 iff clover64");
  }
  REQUIRE(comm->send_lo && comm->send_hi && comm->recv_lo && comm->recv_hi && comm->scalars, "lqcd_cg_solve_slab: NULL comm buffer");
  REQUIRE(comm->exchange_start && comm->exchange_wait && comm->allreduce_sum, "lqcd_cg_solve_slab: NULL callback");
  memset(info, 0, sizeof(*info));
  auto t0 = std::chrono::steady_clock::now();
  const Geom& g = h->g;
  cudaStream_t s = as_stream(stream);
  Workspace ws{(char*)workspace, 0};
  const size_t sites = (size_t)2 * g.Vh;
  void *v64[WS_SPINORS64], *v32[WS_SPINORS32];
  for (int i = 0; i < WS_SPINORS64; i++) v64[i] = ws.take(sites * 12 * sizeof(double2));
  for (int i = 0; i < WS_SPINORS32; i++) v32[i] = ws.take(sites * 12 * sizeof(float2));
  double* partial = (double*)ws.take(partial_len(g) * sizeof(double));
  ws.take(64);
  CgState* state = (CgState*)ws.take(sizeof(CgState));
  const size_t n = spinor_complex(g);
  SlabSolve<double> S{h, d, f->U64, f->clover64, (int)recon, comm, partial, s};
  void *r = v64[0], *p = v64[1], *t = v64[2], *q = v64[3], *bp = v64[4];
  const int check = parm->check_every > 0 ? parm->check_every : 16;
  CgState hs;
  memset(&hs, 0, sizeof(hs));
  double rho0 = 0;
  bool converged = false;

  LSS(S.apply(b, bp, true));                                   // b' = D^+ b
  if (!parm->mixed) {
    LSS(S.cg(bp, x, r, p, t, q, state, parm->tol, parm->maxiter, check, &hs));
    info->iters = hs.iters;
    rho0 = hs.rho0;
    if (hs.breakdown) { set_error("lqcd_cg_solve_slab: breakdown (NaN or <p,D^+D p> <= 0) at iteration %d", hs.iters); return LQCD_EBREAKDOWN; }
    converged = hs.done != 0;
  } else {
    // defect correction as in lqcd_cg_solve: r = b' - D^+D x (fp64); e = CG32(r) to inner_tol; x += e
    SlabSolve<float> S32{h, d, f->U32, f->clover32, (int)recon, comm, partial, s};
    double rho = 0;
    int total = 0;
    const double inner_tol = parm->inner_tol > 0 ? parm->inner_tol : 1e-4;
    CKS(cudaMemsetAsync(x, 0, n * sizeof(double2), s), "memset");
    CKS(cudaMemcpyAsync(r, bp, n * sizeof(double2), cudaMemcpyDeviceToDevice, s), "copy");
    LSS(S.norm2(r, n, &rho0));
    rho = rho0;
    for (;;) {
      if (rho0 == 0.0 || rho <= parm->tol * parm->tol * rho0) { converged = true; break; }
      if (!(rho == rho)) { info->iters = total; set_error("lqcd_cg_solve_slab: NaN residual in mixed solve"); return LQCD_EBREAKDOWN; }
      if (total >= parm->maxiter) break;
      CKS(to_f32(r, v32[0], n, s), "to_f32");
      const double need = parm->tol * sqrt(rho0 / rho) * 0.5;
      const double itol = inner_tol > need ? inner_tol : need;
      LSS(S32.cg(v32[0], v32[5], v32[1], v32[2], v32[3], v32[4], state, itol, parm->maxiter - total, check, &hs));
      total += hs.iters;
      info->outer += 1;
      if (hs.breakdown) { info->iters = total; set_error("lqcd_cg_solve_slab: breakdown in the fp32 inner solve"); return LQCD_EBREAKDOWN; }
      CKS(add_f32_to_f64(v32[5], x, n, s), "x += e");
      LSS(S.apply(x, t, false));
      LSS(S.apply(t, q, true));
      CKS(xmy<double>(bp, q, r, n, s), "r = b' - q");
      LSS(S.norm2(r, n, &rho));
    }
    info->iters = total;
  }
  // true residuals with fresh operator applications (R11), norms over the whole lattice
  double nb = 0, nr = 0, nq = 0;
  LSS(S.apply(x, t, false));
  CKS(xmy<double>(b, t, t, n, s), "b - Dx");
  LSS(S.norm2(b, n, &nb));
  LSS(S.norm2(t, n, &nr));
  LSS(S.apply(t, q, true));
  LSS(S.norm2(q, n, &nq));
  info->rel_resid_true = nb > 0 ? sqrt(nr / nb) : 0.0;
  info->rel_resid_normal = rho0 > 0 ? sqrt(nq / rho0) : 0.0;
  info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  if (!converged) { set_error("lqcd_cg_solve_slab: not converged after %d iterations", info->iters); return LQCD_ENOTCONV; }
  return LQCD_OK;
}

extern "C" {
lqcd_status lqcd_propagator(const lqcd_geom* h, const lqcd_dirac* d, const lqcd_cg_fields* f, const int y[4], void* columns,
                            void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info infos[12], lqcd_recon recon, void* stream) {
  REQUIRE(h && d && f && y && columns && workspace && parm && infos, "lqcd_propagator: NULL argument");
  DeviceGuard dg(h);
  const size_t sbytes = lqcd_field_bytes(h, LQCD_FIELD_SPINOR, LQCD_F64, recon);
  // the source lives in the last fp64 workspace vector, which lqcd_cg_solve does not touch
  void* b = (char*)workspace + (size_t)(WS_SPINORS64 - 1) * align256(sbytes);
  for (int col = 0; col < 12; col++) {
    lqcd_status st = lqcd_point_source(h, y, col / 3, col % 3, b, LQCD_F64, stream);
    if (st != LQCD_OK) return st;
    st = lqcd_cg_solve(h, d, f, b, (char*)columns + (size_t)col * sbytes, workspace, parm, &infos[col], recon, stream);
    if (st != LQCD_OK) return st;
  }
  return LQCD_OK;
}


// ---- several columns in lock step (SURVEY.md 8(f) NEXT-1 carried into the solver) ----------------------------------
static size_t multi_partial_len(const Geom& g, int nrhs) {
  size_t per = (size_t)g.ntiles;
  const size_t np = (size_t)reduce_blocks_max();
  if (np > per) per = np;
  return (size_t)nrhs * per + 64;
}
size_t lqcd_cg_multi_workspace_bytes(const lqcd_geom* h, int nrhs) {
  if (!h || nrhs < 1 || nrhs > 64) return 0;
  const Geom& g = h->g;
  const size_t sp64 = align256((size_t)2 * g.Vh * 12 * sizeof(double2));
  size_t multi = (size_t)4 * nrhs * sp64 + align256(multi_partial_len(g, nrhs) * sizeof(double)) + align256(64) +
                 align256((size_t)nrhs * sizeof(CgState)) + align256(2 * sizeof(int)) + 4096;
  const size_t single = lqcd_field_bytes(h, LQCD_FIELD_WORKSPACE, LQCD_F64, LQCD_RECON_18);
  return multi > single ? multi : single;
}

lqcd_status lqcd_cg_solve_multi(const lqcd_geom* h, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b, void* x,
                                int nrhs, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* infos, lqcd_recon recon,
                                void* stream) {
  REQUIRE(h && d && f && b && x && workspace && parm && infos, "lqcd_cg_solve_multi: NULL argument");
  REQUIRE(good_kappa(d), "lqcd_cg_solve_multi: kappa must be positive and finite (got %g)", d->kappa);
  REQUIRE(nrhs >= 1 && nrhs <= 64, "lqcd_cg_solve_multi: nrhs must be in 1..64");
  REQUIRE(valid_recon(recon), "lqcd_cg_solve_multi: bad recon");
  REQUIRE(f->U64, "lqcd_cg_solve_multi: U64 is required");
  REQUIRE(parm->tol > 0 && parm->maxiter >= 0, "lqcd_cg_solve_multi: bad tol / maxiter");
  UNSUPPORTED_ON_SLAB(h, "lqcd_cg_solve_multi");
  DeviceGuard dg(h);
  const Geom& g = h->g;
  const size_t fb = lqcd_field_bytes(h, LQCD_FIELD_SPINOR, LQCD_F64, recon);
  {
    const char *ib = (const char*)b, *ob = (const char*)x;
    REQUIRE(ob + (size_t)nrhs * fb <= ib || ib + (size_t)nrhs * fb <= ob, "lqcd_cg_solve_multi: b and x overlap");
  }
  SolveCtx c;
  c.h = h; c.d = d; c.f = f; c.parm = parm; c.recon = (int)recon; c.s = as_stream(stream);
  Op<double> M = make_op<double>(c, nullptr);
  M.eo = false;
  if (parm->eo || parm->mixed || nrhs == 1 || !M.multi_fused_ok()) {
    // even-odd / mixed solves, and lattices the pipeline kernel does not serve: one column after the other
    for (int n = 0; n < nrhs; n++) {
      lqcd_status st = lqcd_cg_solve(h, d, f, (const char*)b + (size_t)n * fb, (char*)x + (size_t)n * fb, workspace, parm, &infos[n],
                                     recon, stream);
      if (st != LQCD_OK) return st;
    }
    return LQCD_OK;
  }
  auto t0 = std::chrono::steady_clock::now();
  cudaStream_t s = c.s;
  const size_t nfull = spinor_complex(g);
  Workspace ws{(char*)workspace, 0};
  const size_t arr = (size_t)nrhs * nfull * sizeof(double2);
  void* r = ws.take(arr);
  void* p = ws.take(arr);
  void* t = ws.take(arr);
  void* bm = ws.take(arr);
  double* partial = (double*)ws.take(multi_partial_len(g, nrhs) * sizeof(double));
  double* scratch = (double*)ws.take(64);
  CgState* states = (CgState*)ws.take((size_t)nrhs * sizeof(CgState));
  int* flags = (int*)ws.take(2 * sizeof(int));
  std::vector<CgState> hs(nrhs);
  memset(infos, 0, (size_t)nrhs * sizeof(*infos));
  if (g.bc != LQCD_BC_PERIODIC) {   // D7: components of b on frozen slices are ignored (as in lqcd_cg_solve)
    CKS(cudaMemcpyAsync(bm, b, arr, cudaMemcpyDeviceToDevice, s), "copy b");
    for (int n = 0; n < nrhs; n++) CKS(mask_frozen<double>(g, (double2*)bm + (size_t)n * nfull, s), "mask");
    b = bm;
  }
  CKS(M.apply_multi(b, t, nrhs, true, s), "D^+ b");   // b' in t: copied into r and p before t is first written
  const int check = parm->check_every > 0 ? parm->check_every : 16;
  CKS(cg_normal_multi<double>(M, nrhs, t, x, r, p, t, partial, states, flags, parm->tol, parm->maxiter, check, hs.data(), s),
      "cg_normal_multi");
  // true residuals with fresh operator applications (R11)
  CKS(M.apply_multi(x, t, nrhs, false, s), "D x");
  for (int n = 0; n < nrhs; n++)
    CKS(xmy<double>((const double2*)b + (size_t)n * nfull, (double2*)t + (size_t)n * nfull, (double2*)t + (size_t)n * nfull, nfull, s), "b - Dx");
  CKS(M.apply_multi(t, p, nrhs, true, s), "D^+ (b - Dx)");
  lqcd_status st = LQCD_OK;
  for (int n = 0; n < nrhs; n++) {
    double nb = 0, nr = 0, nq = 0;
    CKS(device_norm2<double>((const double2*)b + (size_t)n * nfull, nfull, partial, scratch, &nb, s), "norm2");
    CKS(device_norm2<double>((const double2*)t + (size_t)n * nfull, nfull, partial, scratch, &nr, s), "norm2");
    CKS(device_norm2<double>((const double2*)p + (size_t)n * nfull, nfull, partial, scratch, &nq, s), "norm2");
    infos[n].iters = hs[n].iters;
    infos[n].rel_resid_true = nb > 0 ? sqrt(nr / nb) : 0.0;
    infos[n].rel_resid_normal = hs[n].rho0 > 0 ? sqrt(nq / hs[n].rho0) : 0.0;
    if (hs[n].breakdown) {
      set_error("lqcd_cg_solve_multi: column %d: breakdown (NaN or <p,M^+M p> <= 0) at iteration %d", n, hs[n].iters);
      st = LQCD_EBREAKDOWN;
    } else if (!hs[n].done && st == LQCD_OK) {
      set_error("lqcd_cg_solve_multi: column %d not converged after %d iterations", n, hs[n].iters);
      st = LQCD_ENOTCONV;
    }
  }
  const double secs = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  for (int n = 0; n < nrhs; n++) infos[n].seconds = secs;
  return st;
}

lqcd_status lqcd_propagator_batched(const lqcd_geom* h, const lqcd_dirac* d, const lqcd_cg_fields* f, const int y[4], void* columns,
                                    void* sources, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info infos[12],
                                    lqcd_recon recon, void* stream) {
  REQUIRE(h && d && f && y && columns && sources && workspace && parm && infos, "lqcd_propagator_batched: NULL argument");
  DeviceGuard dg(h);
  const size_t sbytes = lqcd_field_bytes(h, LQCD_FIELD_SPINOR, LQCD_F64, recon);
  for (int col = 0; col < 12; col++) {
    lqcd_status st = lqcd_point_source(h, y, col / 3, col % 3, (char*)sources + (size_t)col * sbytes, LQCD_F64, stream);
    if (st != LQCD_OK) return st;
  }
  return lqcd_cg_solve_multi(h, d, f, sources, columns, 12, workspace, parm, infos, recon, stream);
}

}  // extern "C"
// ---- host-buffer path -----------------------------------------------------------------------------------------
// Device scratch, streams and the geometry of the last lqcd_dw_apply_host call are kept (one context per process,
// guarded by a mutex) and reused when the next call has the same lattice, precision and link format: seven
// cudaMalloc / cudaFree pairs and a geometry build per call otherwise cost tens of milliseconds.
// lqcd_host_cache_release() frees them.
namespace {
struct HostCtx {
  bool valid = false;
  lqcd_geom_desc desc;
  lqcd_prec prec;
  lqcd_recon recon;
  bool with_clover = false;
  lqcd_geom* h = nullptr;
  void *stage[2] = {nullptr, nullptr}, *dSc = nullptr, *dU64 = nullptr, *dU = nullptr, *dA = nullptr, *dIn = nullptr, *dOut = nullptr;
  cudaStream_t s_copy = nullptr, s_comp = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_spinor = nullptr;
  int slab = 0;   // time slices per staged chunk
  void release() {
    if (!valid && !h) return;
    DeviceGuard dg(desc.device);
    cudaDeviceSynchronize();
    for (int i = 0; i < 2; i++) {
      if (ev_copied[i]) cudaEventDestroy(ev_copied[i]);
      if (ev_free[i]) cudaEventDestroy(ev_free[i]);
      cudaFree(stage[i]);
      ev_copied[i] = ev_free[i] = nullptr; stage[i] = nullptr;
    }
    if (ev_spinor) cudaEventDestroy(ev_spinor);
    if (s_copy) cudaStreamDestroy(s_copy);
    if (s_comp) cudaStreamDestroy(s_comp);
    cudaFree(dSc); cudaFree(dU64); if (dU != dU64) cudaFree(dU); cudaFree(dA); cudaFree(dIn); cudaFree(dOut);
    dSc = dU64 = dU = dA = dIn = dOut = nullptr;
    ev_spinor = nullptr; s_copy = s_comp = nullptr;
    lqcd_geom_destroy(h);
    h = nullptr;
    valid = false;
  }
};
HostCtx g_host;
std::mutex g_host_mutex;


bool same_desc(const lqcd_geom_desc& a, const lqcd_geom_desc& b) {
  bool same = a.bc == b.bc && a.device == b.device && a.slab_edges == b.slab_edges;
  for (int i = 0; i < 4; i++) same = same && a.L[i] == b.L[i] && a.theta[i] == b.theta[i];
  for (int i = 0; i < 3; i++) same = same && a.phi0[i] == b.phi0[i] && a.phiT[i] == b.phiT[i];
  return same;
}
}  // namespace

extern "C" lqcd_status lqcd_host_cache_release(void) {
  std::lock_guard<std::mutex> lock(g_host_mutex);
  g_host.release();
  return LQCD_OK;
}

// The gauge field arrives in time slabs: while slab k + 1 crosses PCIe into one of two staging buffers, slab k is
// converted to the internal layout and the clover term of every time slice whose neighbours are complete is built,
// so that after the last byte of the field only one slab's import, two slices of Csw!, the operator, the export and
// the copy back remain.  The spinor follows the gauge field on the copy stream (same PCIe direction).
extern "C" lqcd_status lqcd_dw_apply_host(const lqcd_geom_desc* desc, const lqcd_dirac* d, const void* U_canon_host,
                                          const void* in_canon_host, void* out_canon_host, int dagger, lqcd_prec prec,
                                          lqcd_recon recon) {
  REQUIRE(desc && d && U_canon_host && in_canon_host && out_canon_host, "lqcd_dw_apply_host: NULL argument");
  REQUIRE(valid_prec(prec) && valid_recon(recon), "lqcd_dw_apply_host: bad precision / recon");
  REQUIRE(desc->bc != LQCD_BC_SLAB, "lqcd_dw_apply_host: a slab needs its neighbours' faces (lqcd_dw_slab_pack / _faces)");
  REQUIRE(good_kappa(d), "lqcd_dw_apply_host: kappa must be positive and finite (got %g)", d->kappa);
  std::lock_guard<std::mutex> lock(g_host_mutex);
  HostCtx& c = g_host;
  const bool with_clover = d->csw != 0.0 || (desc->bc != LQCD_BC_PERIODIC && d->ct != 1.0);
#define HTRY(e, what) do { if (!cuda_ok((e), what)) { c.release(); return LQCD_ECUDA; } } while (0)
#define LTRY(e) do { lqcd_status _s = (e); if (_s != LQCD_OK) { c.release(); return _s; } } while (0)
  if (!(c.valid && !g_host_slab_changed && same_desc(c.desc, *desc) && c.prec == prec && c.recon == recon && c.with_clover == with_clover)) {
    c.release();
    lqcd_status st = lqcd_geom_create(desc, &c.h);
    if (st != LQCD_OK) return st;
    c.desc = *desc; c.prec = prec; c.recon = recon; c.with_clover = with_clover;
    DeviceGuard dg(desc->device);
    const Geom& g = c.h->g;
    const size_t V3 = (size_t)g.L[0] * g.L[1] * g.L[2];
    // slab: a whole number of slices, about 1/12 of the field but not below 64 MB (a copy that short does not reach
    // the link's bandwidth) and not more than the lattice
    int slab = (g.L[3] + 11) / 12;
    while ((size_t)slab * V3 * 36 * sizeof(double2) < ((size_t)64 << 20) && slab < g.L[3]) slab++;
    if (g_host_slab_opt > 0) slab = g_host_slab_opt < g.L[3] ? g_host_slab_opt : g.L[3];   // lqcd_set_option("host_slab")
    g_host_slab_changed = false;
    c.slab = slab;
    HTRY(cudaMalloc(&c.stage[0], (size_t)slab * V3 * 36 * sizeof(double2)), "cudaMalloc");
    HTRY(cudaMalloc(&c.stage[1], (size_t)slab * V3 * 36 * sizeof(double2)), "cudaMalloc");
    HTRY(cudaMalloc(&c.dSc, (size_t)2 * g.Vh * 12 * sizeof(double2)), "cudaMalloc");
    HTRY(cudaMalloc(&c.dU64, lqcd_field_bytes(c.h, LQCD_FIELD_GAUGE, LQCD_F64, recon)), "cudaMalloc");
    if (prec == LQCD_F64) c.dU = c.dU64;
    else HTRY(cudaMalloc(&c.dU, lqcd_field_bytes(c.h, LQCD_FIELD_GAUGE, LQCD_F32, recon)), "cudaMalloc");
    if (with_clover) HTRY(cudaMalloc(&c.dA, lqcd_field_bytes(c.h, LQCD_FIELD_CLOVER, prec, recon)), "cudaMalloc");
    HTRY(cudaMalloc(&c.dIn, lqcd_field_bytes(c.h, LQCD_FIELD_SPINOR, prec, recon)), "cudaMalloc");
    HTRY(cudaMalloc(&c.dOut, lqcd_field_bytes(c.h, LQCD_FIELD_SPINOR, prec, recon)), "cudaMalloc");
    HTRY(cudaStreamCreate(&c.s_copy), "cudaStreamCreate");
    HTRY(cudaStreamCreate(&c.s_comp), "cudaStreamCreate");
    for (int i = 0; i < 2; i++) {
      HTRY(cudaEventCreateWithFlags(&c.ev_copied[i], cudaEventDisableTiming), "cudaEventCreate");
      HTRY(cudaEventCreateWithFlags(&c.ev_free[i], cudaEventDisableTiming), "cudaEventCreate");
    }
    HTRY(cudaEventCreateWithFlags(&c.ev_spinor, cudaEventDisableTiming), "cudaEventCreate");
    c.valid = true;
  }
  DeviceGuard dg(desc->device);
  const lqcd_geom* h = c.h;
  const Geom& g = h->g;
  const size_t V3 = (size_t)g.L[0] * g.L[1] * g.L[2];
  const size_t slice_bytes = V3 * 36 * sizeof(double2);
  const size_t sc = (size_t)2 * g.Vh * 12 * sizeof(double2);
  CloverParm cp;
  cp.kappa = d->kappa; cp.csw = d->csw; cp.ct = d->ct;
  for (int i = 0; i < 3; i++) cp.phiT[i] = desc->phiT[i];
  int built = 1;   // slices [1, built) of the clover term are done (slice 0 needs the last slice: at the end)
  int k = 0;
  for (int t0 = 0; t0 < g.L[3]; t0 += c.slab, k++) {
    const int t1 = t0 + c.slab < g.L[3] ? t0 + c.slab : g.L[3];
    const int b = k & 1;
    if (k >= 2) HTRY(cudaStreamWaitEvent(c.s_copy, c.ev_free[b], 0), "wait");
    HTRY(cudaMemcpyAsync(c.stage[b], (const char*)U_canon_host + (size_t)t0 * slice_bytes, (size_t)(t1 - t0) * slice_bytes,
                         cudaMemcpyHostToDevice, c.s_copy), "H2D gauge slab");
    HTRY(cudaEventRecord(c.ev_copied[b], c.s_copy), "event");
    HTRY(cudaStreamWaitEvent(c.s_comp, c.ev_copied[b], 0), "wait");
    HTRY(gauge_import_slab<double>(g, c.stage[b], c.dU64, (int)recon, t0, t1, c.s_comp), "gauge_import (slab)");
    if (prec == LQCD_F32) HTRY(gauge_import_slab<float>(g, c.stage[b], c.dU, (int)recon, t0, t1, c.s_comp), "gauge_import (slab)");
    HTRY(cudaEventRecord(c.ev_free[b], c.s_comp), "event");
    if (with_clover && t1 - 1 > built) {   // slices below t1 - 1 have both time neighbours on the device
      cp.t_lo = built; cp.t_hi = t1 - 1;
      HTRY(clover_build(g, cp, c.dU64, (int)recon, c.dA, nullptr, (int)prec, c.s_comp), "clover_build (slab)");
      built = t1 - 1;
    }
  }
  HTRY(cudaMemcpyAsync(c.dSc, in_canon_host, sc, cudaMemcpyHostToDevice, c.s_copy), "H2D spinor");
  HTRY(cudaEventRecord(c.ev_spinor, c.s_copy), "event");
  if (with_clover) {
    cp.t_lo = built; cp.t_hi = g.L[3];
    HTRY(clover_build(g, cp, c.dU64, (int)recon, c.dA, nullptr, (int)prec, c.s_comp), "clover_build (last slices)");
    cp.t_lo = 0; cp.t_hi = 1;
    HTRY(clover_build(g, cp, c.dU64, (int)recon, c.dA, nullptr, (int)prec, c.s_comp), "clover_build (slice 0)");
  }
  HTRY(cudaStreamWaitEvent(c.s_comp, c.ev_spinor, 0), "wait");
  LTRY(lqcd_spinor_import(h, c.dSc, c.dIn, prec, c.s_comp));
  LTRY(dw_common(h, d, c.dU, with_clover ? c.dA : nullptr, c.dIn, c.dOut, prec, recon, c.s_comp, dagger != 0));
  LTRY(lqcd_spinor_export(h, c.dOut, c.dSc, prec, c.s_comp));
  HTRY(cudaMemcpyAsync(out_canon_host, c.dSc, sc, cudaMemcpyDeviceToHost, c.s_comp), "D2H spinor");
  HTRY(cudaStreamSynchronize(c.s_comp), "sync");
  HTRY(cudaStreamSynchronize(c.s_copy), "sync");
#undef HTRY
#undef LTRY
  return LQCD_OK;
}


// ---------------------------------------------------------------------------------------------------------------
// SU(2) fundamental representation
// ---------------------------------------------------------------------------------------------------------------
namespace {
bool su2_bc_ok(const lqcd_geom* h) { return h->g.bc == LQCD_BC_PERIODIC || h->g.bc == LQCD_BC_OPEN; }
size_t su2_spinor_complex(const Geom& g) { return (size_t)2 * g.Vh * 8; }
}  // namespace
#define SU2_COMMON(h, d, name)                                                                                      \
  do {                                                                                                             \
    REQUIRE(su2_bc_ok(h), name ": SU(2) fields support periodic and open time boundaries only");                  \
    if (d) {                                                                                                       \
      REQUIRE(good_kappa((const lqcd_dirac*)(d)), name ": kappa must be positive and finite");                    \
      REQUIRE(((const lqcd_dirac*)(d))->mu == 0.0 && ((const lqcd_dirac*)(d))->ct == 1.0, name ": mu = 0 and ct = 1 only in the SU(2) representation"); \
    }                                                                                                              \
  } while (0)

extern "C" {

size_t lqcd_su2_field_bytes(const lqcd_geom* h, lqcd_field_kind kind, lqcd_prec prec) {
  if (!h) return 0;
  const Geom& g = h->g;
  const size_t sites = (size_t)2 * g.Vh, eb = elem_bytes(prec);
  switch (kind) {
    case LQCD_FIELD_GAUGE: return sites * 8 * eb;
    case LQCD_FIELD_SPINOR: return sites * 8 * eb;
    case LQCD_FIELD_CLOVER: return sites * 16 * eb;
    case LQCD_FIELD_WORKSPACE: return 6 * align256(sites * 8 * sizeof(double2)) + 2 * align256(partial_len(g) * sizeof(double)) + 4096;
    default: return 0;
  }
}
lqcd_status lqcd_su2_gauge_import(const lqcd_geom* h, const void* canon, void* U, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && U && canon != U, "lqcd_su2_gauge_import: NULL or aliased argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_gauge_import: bad precision");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_gauge_import<double>(h->g, canon, U, as_stream(stream)), su2_gauge_import<float>(h->g, canon, U, as_stream(stream))), "su2_gauge_import");
  return LQCD_OK;
}
lqcd_status lqcd_su2_gauge_export(const lqcd_geom* h, const void* U, void* canon, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && U && canon != U, "lqcd_su2_gauge_export: NULL or aliased argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_gauge_export: bad precision");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_gauge_export<double>(h->g, U, canon, as_stream(stream)), su2_gauge_export<float>(h->g, U, canon, as_stream(stream))), "su2_gauge_export");
  return LQCD_OK;
}
lqcd_status lqcd_su2_spinor_import(const lqcd_geom* h, const void* canon, void* psi, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && psi && canon != psi, "lqcd_su2_spinor_import: NULL or aliased argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_spinor_import: bad precision");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_spinor_import<double>(h->g, canon, psi, as_stream(stream)), su2_spinor_import<float>(h->g, canon, psi, as_stream(stream))), "su2_spinor_import");
  return LQCD_OK;
}
lqcd_status lqcd_su2_spinor_export(const lqcd_geom* h, const void* psi, void* canon, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && psi && canon != psi, "lqcd_su2_spinor_export: NULL or aliased argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_spinor_export: bad precision");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_spinor_export<double>(h->g, psi, canon, as_stream(stream)), su2_spinor_export<float>(h->g, psi, canon, as_stream(stream))), "su2_spinor_export");
  return LQCD_OK;
}
lqcd_status lqcd_su2_clover_build(const lqcd_geom* h, const lqcd_dirac* d, const void* U64, void* clover, lqcd_prec out_prec, void* stream) {
  REQUIRE(h && d && U64 && clover && clover != U64, "lqcd_su2_clover_build: NULL or aliased argument");
  REQUIRE(valid_prec(out_prec), "lqcd_su2_clover_build: bad precision");
  SU2_COMMON(h, d, "lqcd_su2_clover_build");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(out_prec, su2_clover_build<double>(h->g, d->kappa, d->csw, U64, clover, as_stream(stream)),
                         su2_clover_build<float>(h->g, d->kappa, d->csw, U64, clover, as_stream(stream))), "su2_clover_build");
  return LQCD_OK;
}
lqcd_status lqcd_su2_clover_export(const lqcd_geom* h, const void* clover, void* canon, lqcd_prec prec, void* stream) {
  REQUIRE(h && canon && clover && canon != clover, "lqcd_su2_clover_export: NULL or aliased argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_clover_export: bad precision");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_clover_export<double>(h->g, clover, canon, as_stream(stream)), su2_clover_export<float>(h->g, clover, canon, as_stream(stream))), "su2_clover_export");
  return LQCD_OK;
}
lqcd_status lqcd_su2_dw_apply(const lqcd_geom* h, const lqcd_dirac* d, const void* U, const void* clover, const void* in, void* out,
                              int dagger, lqcd_prec prec, void* stream) {
  REQUIRE(h && d && U && in && out, "lqcd_su2_dw_apply: NULL argument");
  REQUIRE(valid_prec(prec), "lqcd_su2_dw_apply: bad precision");
  REQUIRE(out != in && out != U && out != clover, "lqcd_su2_dw_apply: output aliases an input");
  SU2_COMMON(h, d, "lqcd_su2_dw_apply");
  DeviceGuard dg(h);
  CUDA_TRY(DISPATCH_PREC(prec, su2_dw<double>(h, d->kappa, U, clover, in, out, dagger != 0, as_stream(stream)),
                         su2_dw<float>(h, d->kappa, U, clover, in, out, dagger != 0, as_stream(stream))), "su2_dw kernel");
  return LQCD_OK;
}

// CG on D^+ D x = D^+ b in fp64 (the algorithm of lqcd_cg_solve, unfused BLAS-1, scalars on the device)
lqcd_status lqcd_su2_cg_solve(const lqcd_geom* h, const lqcd_dirac* d, const void* U64, const void* clover64, const void* b, void* x,
                              void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info, void* stream) {
  REQUIRE(h && d && U64 && b && x && workspace && parm && info, "lqcd_su2_cg_solve: NULL argument");
  REQUIRE(x != b, "lqcd_su2_cg_solve: x aliases b");
  REQUIRE(parm->tol > 0 && parm->maxiter >= 0 && !parm->eo && !parm->mixed, "lqcd_su2_cg_solve: bad tol / maxiter, or eo / mixed (not available for SU(2))");
  SU2_COMMON(h, d, "lqcd_su2_cg_solve");
  DeviceGuard dg(h);
  memset(info, 0, sizeof(*info));
  auto t0 = std::chrono::steady_clock::now();
  const Geom& g = h->g;
  cudaStream_t s = as_stream(stream);
  const size_t n = su2_spinor_complex(g), bytes = n * sizeof(double2);
  Workspace ws{(char*)workspace, 0};
  void *r = ws.take(bytes), *p = ws.take(bytes), *t = ws.take(bytes), *q = ws.take(bytes), *bp = ws.take(bytes), *bm = ws.take(bytes);
  double* partial = (double*)ws.take(partial_len(g) * sizeof(double));
  double* scratch = (double*)ws.take(64);
  CgState* state = (CgState*)ws.take(sizeof(CgState));
  const int nb = reduce_blocks(n);
  auto D = [&](const void* in, void* out, bool dag) { return su2_dw<double>(h, d->kappa, U64, clover64, in, out, dag, s); };
  CKS(cudaMemcpyAsync(bm, b, bytes, cudaMemcpyDeviceToDevice, s), "copy b");
  if (g.bc != LQCD_BC_PERIODIC) CKS(su2_mask_frozen<double>(g, bm, s), "mask");   // D7: the solve lives on the interior
  CKS(D(bm, bp, true), "D^+ b");
  CKS(cudaMemsetAsync(x, 0, bytes, s), "memset");
  CKS(cudaMemcpyAsync(r, bp, bytes, cudaMemcpyDeviceToDevice, s), "copy");
  CKS(cudaMemcpyAsync(p, bp, bytes, cudaMemcpyDeviceToDevice, s), "copy");
  CKS(norm2_partial<double>(r, n, partial, s), "norm2");
  CKS(cg_init_state(state, partial, nb, parm->tol, s), "cg_init_state");
  const int check = parm->check_every > 0 ? parm->check_every : 16;
  CgState hs;
  int launched = 0;
  for (;;) {
    CKS(cudaMemcpyAsync(&hs, state, sizeof(CgState), cudaMemcpyDeviceToHost, s), "copy state");
    CKS(cudaStreamSynchronize(s), "sync");
    if (hs.done || launched >= parm->maxiter) break;
    int batch = check;
    if (launched + batch > parm->maxiter) batch = parm->maxiter - launched;
    for (int it = 0; it < batch; it++) {
      CKS(D(p, t, false), "D p");
      CKS(norm2_partial<double>(t, n, partial, s), "norm2");
      CKS(cg_reduce_alpha(state, partial, nb, s), "alpha");
      CKS(D(t, q, true), "D^+ t");
      CKS(cg_raxpy_norm<double>(state, q, r, n, partial, s), "r -= alpha q");
      CKS(cg_reduce_beta(state, partial, nb, s), "beta");
      CKS(cg_update_xp<double>(state, x, p, r, n, s), "update");
    }
    launched += batch;
  }
  info->iters = hs.iters;
  // true residuals with fresh operator applications (R11)
  double nbv = 0, nr = 0, nq = 0;
  CKS(D(x, t, false), "D x");
  CKS(xmy<double>(bm, t, t, n, s), "b - Dx");
  CKS(device_norm2<double>(bm, n, partial, scratch, &nbv, s), "norm2");
  CKS(device_norm2<double>(t, n, partial, scratch, &nr, s), "norm2");
  CKS(D(t, q, true), "D^+ (b - Dx)");
  CKS(device_norm2<double>(q, n, partial, scratch, &nq, s), "norm2");
  info->rel_resid_true = nbv > 0 ? sqrt(nr / nbv) : 0.0;
  info->rel_resid_normal = hs.rho0 > 0 ? sqrt(nq / hs.rho0) : 0.0;
  info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  if (hs.breakdown) { set_error("lqcd_su2_cg_solve: breakdown (NaN or <p,D^+D p> <= 0) at iteration %d", hs.iters); return LQCD_EBREAKDOWN; }
  if (!hs.done) { set_error("lqcd_su2_cg_solve: not converged after %d iterations", hs.iters); return LQCD_ENOTCONV; }
  return LQCD_OK;
}

}  // extern "C"
