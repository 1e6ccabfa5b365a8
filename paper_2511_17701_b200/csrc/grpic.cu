// grpic.cu — host side of the C ABI declared in include/grpic.h: argument checks, context,
// launches.  One source, two builds (-DGRPIC_F64 selects grpic_real = double).
// There is no CPU fallback anywhere in this file: every compute entry point launches CUDA kernels
// or returns an error.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "../../include/grpic.h"
#include "grpic_kernels.cuh"
#include "grpic_tiled.cuh"
#include "grpic_lanes.cuh"
#include "grpic_fields.cuh"
#include "grpic_probe.cuh"

using namespace grpic;
typedef grpic_real real;

namespace {

std::string g_create_error;

struct SortState {          // tile table of one species (keyed by the address of its i1 column)
  int64_t n_at_sort = 0;    // p->n when the table was built
  // Alive particles at that time, d_n_items[1] on the device: slots [0, n_alive) are covered by the table, the rest
  // (dead at sort time, or appended later) by the direct path, so revived / injected particles are never skipped.
  // The host copy is fetched only when somebody asks (grpic_sorted_alive, or a call with p->n < n_at_sort).
  int64_t n_alive = 0;
  bool n_alive_known = false;
  cudaStream_t stream = nullptr;   // stream of the sort (the read-back waits on it)
  uint64_t stamp = 0;              // ctx->stamp at the last sort: the oldest table goes when there are too many
  WorkItem* items = nullptr;
  uint32_t* d_n_items = nullptr;   // [0] items, [1] alive particles at sort time, [2] dense items
  uint32_t* dense_idx = nullptr;   // indices of the dense items (k_step_lanes), [max_items]
  uint32_t* offsets = nullptr;     // scanned key histogram of the last sort (n_keys + 1): first slot of every sort key
  uint32_t max_items = 0;
  uint32_t max_dense = 0;          // upper bound of [2]: grid of k_step_lanes
};

}  // namespace

struct grpic_ctx {
  grpic_grid grid;
  double a, r_min, r_max, small_angle, r0, h0, mass, k_J;
  int n_iter, tile_path, use_tma, early_exit;
  int lanes_path;           // 1: dense work items go to k_step_lanes (grpic_lanes.cuh)
  int64_t dense_min;        // particles from which a work item counts as dense
  // dynamic shared-memory opt-in done on ctx->device for: k_step_lanes<real, Coord / CoordGen>,
  // k_step_tiled<real, Coord / CoordGen, push-only / fused>, k_deposit_tiled<real, Coord / CoordGen>
  bool lanes_attr[2], tiled_attr[2][2], dep_attr[2];
  // side stream of grpic_step (sparse items and tail slots beside k_step_lanes)
  int overlap;
  bool side_ok;
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_join;
  int64_t host_chunk;       // particles per chunk of grpic_step_host
  double sort_lookahead;    // steps of the last dt the sort key looks ahead (0 = present cell)
  double last_dt;
  bool have_dt;
  unsigned long long* d_counters;   // 5: four of the last call + cumulative updates
  std::string err;
  int device;
  // sort scratch
  uint32_t *d_keys, *d_dest, *d_hist, *d_block_sums, *d_tile_items;
  int64_t cap_particles;
  void* d_scratch;
  size_t scratch_bytes;
  std::map<const void*, SortState> sorted;   // at most kMaxTables entries (grpic_forget drops one; the oldest is evicted)
  uint64_t stamp;
  // TMA
  TmaEncoder tma;
  // grpic_step_host buffers
  void* h_dev[16];
  size_t h_cap;
  void* h_fields;
  size_t h_fields_bytes;
  cudaStream_t h_streams[3];
  real* f_scratch;          // 12 grid arrays for the field side of the PIC loop: E[3] H[3] Dh[3] Jn[3]
  size_t f_scratch_cells;
  bool h_streams_ok;
};

namespace {

int fail(grpic_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}
int cuda_fail(grpic_ctx* c, cudaError_t e, const char* what) {
  return fail(c, GRPIC_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);  \
  } while (0)

// Every buffer, the tile tables and the shared-memory opt-ins of a context belong to the device that was current at
// grpic_create: a call made with another device current is refused rather than launched on the wrong GPU.
int check_device(grpic_ctx* ctx) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device)
    return fail(ctx, GRPIC_ESTATE, "the current CUDA device is not the one this context was created on");
  return GRPIC_OK;
}

Consts<real> make_consts(const grpic_ctx* c) {
  Consts<real> g;
  g.n1 = c->grid.n1; g.n2 = c->grid.n2; g.ng = c->grid.nghost; g.n_iter = c->n_iter;
  g.ld = c->grid.n2 + 2 * c->grid.nghost;
  const bool lin = c->grid.r_map == 0;             // A.2: dxi = 1 and rm = dr make s1 = dxi*rm = dr (grpic_device.cuh)
  const double dxi = lin ? 1.0 : std::log((c->r_max - c->r0) / (c->r_min - c->r0)) / c->grid.n1;
  const double deta = M_PI / c->grid.n2;
  g.r_lin = lin ? 1 : 0;
  g.r_min = (real)c->r_min;
  g.dr = (real)((c->r_max - c->r_min) / c->grid.n1);
  g.dls1 = lin ? (real)0 : (real)dxi;
  g.a = (real)c->a; g.a2 = (real)(c->a * c->a);
  g.log_rmin = lin ? (real)0 : (real)std::log(c->r_min - c->r0);
  g.r_off = (real)c->r0; g.h0 = (real)c->h0; g.mass = (real)c->mass;
  g.dxi = (real)dxi; g.deta = (real)deta;
  g.inv_dxi = (real)(1.0 / dxi);
  g.inv_deta2 = (real)(1.0 / (deta * deta));
  g.th_min = (real)c->small_angle;
  g.th_max = (real)(M_PI - c->small_angle);
  g.sin_min = (real)std::sin((double)g.th_min);
  g.cos_min = (real)std::cos((double)g.th_min);
  g.sin_max = (real)std::sin((double)g.th_max);
  g.cos_max = (real)std::cos((double)g.th_max);
  g.early_exit = c->early_exit;
  return g;
}

PPtrs<real> make_pptrs(const grpic_particles* p) {
  PPtrs<real> P;
  P.n = p->n;
  P.i1 = p->i1; P.i2 = p->i2; P.dx1 = p->dx1; P.dx2 = p->dx2;
  P.u1 = p->u1; P.u2 = p->u2; P.u3 = p->u3; P.phi = p->phi;
  P.i1p = p->i1_prev; P.i2p = p->i2_prev; P.dx1p = p->dx1_prev; P.dx2p = p->dx2_prev;
  P.w = p->weight; P.tag = p->tag;
  return P;
}

// need_prev: 0 = the *_prev columns are not looked at, 1 = required, 2 = all four or none
int check_particles(grpic_ctx* ctx, const grpic_particles* p, int need_prev) {
  if (!p) return fail(ctx, GRPIC_EINVAL, "particles == NULL");
  if (p->n < 0) return fail(ctx, GRPIC_EINVAL, "particles.n < 0");
  if (p->n > 0xfffffff0ll) return fail(ctx, GRPIC_EINVAL, "particles.n exceeds 2^32 - 16");
  if (p->n == 0) return GRPIC_OK;
  if (!p->i1 || !p->i2 || !p->dx1 || !p->dx2 || !p->u1 || !p->u2 || !p->u3 || !p->weight || !p->tag)
    return fail(ctx, GRPIC_EINVAL, "a required particle column is NULL");
  const int n_prev = (p->i1_prev != nullptr) + (p->i2_prev != nullptr) + (p->dx1_prev != nullptr) + (p->dx2_prev != nullptr);
  if (need_prev == 1 && n_prev != 4) return fail(ctx, GRPIC_EINVAL, "a *_prev particle column is NULL");
  if (need_prev == 2 && n_prev != 4 && n_prev != 0)
    return fail(ctx, GRPIC_EINVAL, "the *_prev particle columns must be all present or all NULL");
  return GRPIC_OK;
}

SpeciesConst make_species(const grpic_particles* p, double dt, bool deposit) {
  SpeciesConst sc;
  sc.q_over_m = p->q_over_m; sc.charge = p->charge; sc.dt = dt;
  sc.massive = p->massive ? 1 : 0;
  sc.em = (p->q_over_m != 0.0 && p->massive) ? 1 : 0;
  sc.has_phi = p->phi ? 1 : 0;
  sc.do_deposit = (deposit && p->charge != 0.0) ? 1 : 0;
  return sc;
}

int check_fields(grpic_ctx* ctx, const grpic_fields* f, const SpeciesConst& sc, FPtrs<real>& F) {
  for (int k = 0; k < 6; ++k) F.f[k] = nullptr;
  if (!sc.em) return GRPIC_OK;
  if (!f) return fail(ctx, GRPIC_EINVAL, "fields == NULL for a charged massive species");
  const real* a[6] = {f->D1, f->D2, f->D3, f->B1, f->B2, f->B3};
  for (int k = 0; k < 6; ++k) {
    if (!a[k]) return fail(ctx, GRPIC_EINVAL, "a field component pointer is NULL");
    F.f[k] = a[k];
  }
  return GRPIC_OK;
}

int check_current(grpic_ctx* ctx, const grpic_current* J, const SpeciesConst& sc, JPtrs<real>& Jp) {
  for (int k = 0; k < 3; ++k) Jp.j[k] = nullptr;
  if (!sc.do_deposit) return GRPIC_OK;
  if (!J || !J->J1 || !J->J2 || !J->J3) return fail(ctx, GRPIC_EINVAL, "current pointers are NULL for a charged species");
  Jp.j[0] = J->J1; Jp.j[1] = J->J2; Jp.j[2] = J->J3;
  return GRPIC_OK;
}

FieldGeom make_field_geom(const grpic_ctx* c) {
  FieldGeom q;
  q.n1 = c->grid.n1; q.n2 = c->grid.n2; q.ng = c->grid.nghost;
  q.ld = c->grid.n2 + 2 * c->grid.nghost; q.rows = c->grid.n1 + 2 * c->grid.nghost;
  q.r_lin = c->grid.r_map == 0 ? 1 : 0;
  q.a = c->a; q.mass = c->mass; q.r_off = c->r0; q.h0 = c->h0;
  q.log_rmin = q.r_lin ? 0.0 : std::log(c->r_min - c->r0);
  q.dxi = q.r_lin ? 1.0 : std::log((c->r_max - c->r0) / (c->r_min - c->r0)) / c->grid.n1;
  q.deta = M_PI / c->grid.n2;
  q.r_min = c->r_min; q.dr = (c->r_max - c->r_min) / c->grid.n1;
  return q;
}

inline bool general_map(const grpic_ctx* c) {
  return c->r0 != 0.0 || c->h0 != 0.0 || c->grid.r_map == 0 || c->mass != 1.0;
}
inline unsigned grid_for(int64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

int scan_exclusive(grpic_ctx* ctx, uint32_t* d, uint32_t n, cudaStream_t st) {
  const uint32_t nb = (n + kScanTile - 1) / kScanTile;
  k_scan_local<<<nb, kScanBlock, 0, st>>>(d, n, ctx->d_block_sums);
  k_scan_sums<<<1, kScanBlock, 0, st>>>(ctx->d_block_sums, nb);
  k_scan_add<<<nb, kScanBlock, 0, st>>>(d, n, ctx->d_block_sums);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

SortGeom sort_geom(const grpic_ctx* c) {
  SortGeom s;
  s.n1 = c->grid.n1; s.n2 = c->grid.n2;
  s.nt1 = (c->grid.n1 + kTile - 1) / kTile;
  s.nt2 = (c->grid.n2 + kTile - 1) / kTile;
  s.n_keys = (uint32_t)s.nt1 * s.nt2 * kTile * kTile + 1u;
  return s;
}

// host copy of the alive count of the last sort (synchronises the stream of that sort, once)
int fetch_alive(grpic_ctx* ctx, SortState& s) {
  if (s.n_alive_known) return GRPIC_OK;
  uint32_t h = 0;
  CK(cudaMemcpyAsync(&h, s.d_n_items + 1, sizeof(uint32_t), cudaMemcpyDeviceToHost, s.stream));
  CK(cudaStreamSynchronize(s.stream));
  s.n_alive = (int64_t)h;
  s.n_alive_known = true;
  return GRPIC_OK;
}

// May the tile table of `s` serve a call on p?  Yes while p still has every slot the table covers: always if p->n has
// not shrunk since the sort; after a compaction (p->n lowered towards the alive count) the count is fetched once.
bool table_covers(grpic_ctx* ctx, SortState& s, const grpic_particles* p) {
  if (p->n >= s.n_at_sort) return true;
  if (fetch_alive(ctx, s) != GRPIC_OK) return false;
  return s.n_alive <= p->n;
}

// grid of the kernels that walk the slots behind the alive count (k_*_from): fixed, block-strided
constexpr unsigned kTailGrid = 148 * 4;

void free_sort_state(SortState& s) {
  if (s.items) cudaFree(s.items);
  if (s.d_n_items) cudaFree(s.d_n_items);
  if (s.dense_idx) cudaFree(s.dense_idx);
  if (s.offsets) cudaFree(s.offsets);
  s = SortState();
}

}  // namespace

extern "C" {

int grpic_real_bytes(void) { return (int)sizeof(real); }
int grpic_tile_size(void) { return kTile; }

const char* grpic_last_error(grpic_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int grpic_create(const grpic_grid* grid, double a, double r_min, double r_max, grpic_ctx** out) {
  grpic_ctx* ctx = nullptr;
  if (!grid || !out) return fail(nullptr, GRPIC_EINVAL, "grid or out is NULL");
  *out = nullptr;
  if (grid->n1 < 1 || grid->n2 < 1) return fail(nullptr, GRPIC_EINVAL, "n1, n2 must be >= 1");
  if (grid->nghost < 1) return fail(nullptr, GRPIC_EINVAL, "nghost must be >= 1 (the gather reads one ghost layer)");
  if (grid->r_map != 0 && grid->r_map != 1)
    return fail(nullptr, GRPIC_EINVAL, "r_map must be 1 (logarithmic r, App. A.3) or 0 (uniform r, App. A.2)");
  if (!(r_min > 0.0) || !(r_max > r_min)) return fail(nullptr, GRPIC_EINVAL, "need 0 < r_min < r_max");
  if (!(std::fabs(a) <= 1.0)) return fail(nullptr, GRPIC_EINVAL, "need |a| <= 1");
  if ((int64_t)(grid->n1 + 2 * grid->nghost) * (grid->n2 + 2 * grid->nghost) > 0x7fffffffll)
    return fail(nullptr, GRPIC_EINVAL, "grid too large");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev < 1)
    return fail(nullptr, GRPIC_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
  ctx = new (std::nothrow) grpic_ctx();
  if (!ctx) return fail(nullptr, GRPIC_ENOMEM, "host allocation failed");
  ctx->grid = *grid;
  ctx->a = a; ctx->r_min = r_min; ctx->r_max = r_max;
  ctx->small_angle = 1e-5;                                  // SMALL_ANGLE_GR
  ctx->r0 = 0.0; ctx->h0 = 0.0;                             // A.3 map parameters
  ctx->mass = 1.0;                                          // r_g = M = 1
  ctx->k_J = 4.0 * M_PI;                                    // coefficient of J in Ampere's law (Eq. 37)
  ctx->n_iter = 10;
  ctx->tile_path = 1;
  ctx->lanes_path = 1;
  ctx->dense_min = 2048;
  ctx->lanes_attr[0] = ctx->lanes_attr[1] = false;
  ctx->tiled_attr[0][0] = ctx->tiled_attr[0][1] = ctx->tiled_attr[1][0] = ctx->tiled_attr[1][1] = false;
  ctx->dep_attr[0] = ctx->dep_attr[1] = false;
  ctx->overlap = 1; ctx->side_ok = false; ctx->side = nullptr; ctx->ev_fork = ctx->ev_join = nullptr;
  ctx->host_chunk = 1 << 22;
  ctx->sort_lookahead = 0.0;
  ctx->use_tma = 1;
  ctx->early_exit = 1;
  ctx->have_dt = false; ctx->last_dt = 0.0;
  ctx->d_counters = nullptr;
  ctx->d_keys = ctx->d_dest = ctx->d_hist = ctx->d_block_sums = ctx->d_tile_items = nullptr;
  ctx->cap_particles = 0;
  ctx->stamp = 0;
  ctx->d_scratch = nullptr; ctx->scratch_bytes = 0;
  for (auto& q : ctx->h_dev) q = nullptr;
  ctx->f_scratch = nullptr; ctx->f_scratch_cells = 0;
  ctx->h_cap = 0; ctx->h_fields = nullptr; ctx->h_fields_bytes = 0; ctx->h_streams_ok = false;
  cudaGetDevice(&ctx->device);
  e = cudaMalloc(&ctx->d_counters, 8 * sizeof(unsigned long long));
  if (e != cudaSuccess) {
    std::string m = std::string("cudaMalloc(counters): ") + cudaGetErrorString(e);
    delete ctx;
    return fail(nullptr, GRPIC_ECUDA, m);
  }
  cudaMemset(ctx->d_counters, 0, 8 * sizeof(unsigned long long));
  ctx->tma.init();
  *out = ctx;
  return GRPIC_OK;
}

int grpic_destroy(grpic_ctx* ctx) {
  if (!ctx) return GRPIC_OK;
  cudaDeviceSynchronize();
  for (auto& kv : ctx->sorted) free_sort_state(kv.second);
  cudaFree(ctx->d_counters);
  cudaFree(ctx->d_keys); cudaFree(ctx->d_dest); cudaFree(ctx->d_hist);
  cudaFree(ctx->d_block_sums); cudaFree(ctx->d_tile_items);
  cudaFree(ctx->d_scratch);
  for (auto q : ctx->h_dev) cudaFree(q);
  cudaFree(ctx->h_fields);
  cudaFree(ctx->f_scratch);
  if (ctx->h_streams_ok) for (auto& q : ctx->h_streams) cudaStreamDestroy(q);
  if (ctx->side_ok) { cudaStreamDestroy(ctx->side); cudaEventDestroy(ctx->ev_fork); cudaEventDestroy(ctx->ev_join); }
  delete ctx;
  return GRPIC_OK;
}

int grpic_set_int(grpic_ctx* ctx, const char* key, int64_t v) {
  if (!ctx || !key) return fail(ctx, GRPIC_EINVAL, "ctx or key is NULL");
  if (!std::strcmp(key, "n_iter")) {
    if (v < 1 || v > 64) return fail(ctx, GRPIC_EINVAL, "n_iter must be in 1..64");
    ctx->n_iter = (int)v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "tile_path")) {
    ctx->tile_path = v ? 1 : 0;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "overlap")) {
    ctx->overlap = v ? 1 : 0;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "lanes_path")) {
    ctx->lanes_path = v ? 1 : 0;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "dense_min")) {
    if (v < 4 || v > kChunk) return fail(ctx, GRPIC_EINVAL, "dense_min must be in 4..16384");
    ctx->dense_min = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "early_exit")) {
    ctx->early_exit = v ? 1 : 0;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "tma")) {
    ctx->use_tma = v ? 1 : 0;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "host_chunk")) {
    if (v < 1024 || v > (1 << 26)) return fail(ctx, GRPIC_EINVAL, "host_chunk must be in 2^10..2^26");
    ctx->host_chunk = v;
    return GRPIC_OK;
  }
  return fail(ctx, GRPIC_EINVAL, std::string("unknown integer key: ") + key);
}

int grpic_set_real(grpic_ctx* ctx, const char* key, double v) {
  if (!ctx || !key) return fail(ctx, GRPIC_EINVAL, "ctx or key is NULL");
  if (!std::strcmp(key, "small_angle")) {
    if (!(v >= 0.0 && v < 1.0)) return fail(ctx, GRPIC_EINVAL, "small_angle must be in [0, 1)");
    ctx->small_angle = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "sort_lookahead")) {
    if (!(v >= 0.0 && v <= 64.0)) return fail(ctx, GRPIC_EINVAL, "sort_lookahead must be in [0, 64]");
    ctx->sort_lookahead = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "r0")) {
    if (!(v < ctx->r_min)) return fail(ctx, GRPIC_EINVAL, "r0 must be < r_min");
    ctx->r0 = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "k_J")) {
    ctx->k_J = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "mass")) {
    if (!(v >= 0.0)) return fail(ctx, GRPIC_EINVAL, "mass must be >= 0");
    ctx->mass = v;
    return GRPIC_OK;
  }
  if (!std::strcmp(key, "h0")) {
    if (!(v > -0.5 && v < 1.0)) return fail(ctx, GRPIC_EINVAL, "h0 must be in (-0.5, 1): dtheta/deta > 0");
    ctx->h0 = v;
    return GRPIC_OK;
  }
  return fail(ctx, GRPIC_EINVAL, std::string("unknown real key: ") + key);
}

int grpic_interp_push(grpic_ctx* ctx, grpic_particles* p, const grpic_fields* fields, double dt, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, p, 1);
  if (rc) return rc;
  if (!(dt > 0.0)) return fail(ctx, GRPIC_EINVAL, "dt must be > 0");
  const SpeciesConst sc = make_species(p, dt, false);
  FPtrs<real> F;
  if ((rc = check_fields(ctx, fields, sc, F))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  ctx->last_dt = dt; ctx->have_dt = true;
  CK(cudaMemsetAsync(ctx->d_counters, 0, 3 * sizeof(unsigned long long), st));
  if (p->n == 0) return GRPIC_OK;
  JPtrs<real> J{{nullptr, nullptr, nullptr}};
  {
    auto it = ctx->sorted.find((const void*)p->i1);
    if (ctx->tile_path && it != ctx->sorted.end() && sc.em && table_covers(ctx, it->second, p)) {
      // sorted species: field stencil of each tile staged in shared memory, as in the fused step
      const SortState& ss = it->second;
      std::string terr;
      const Consts<real> g = make_consts(ctx);
      const PPtrs<real> P = make_pptrs(p);
      const bool ok = general_map(ctx)
          ? launch_step_tiled<real, CoordGen<real>, false>(ctx->tma, ctx->use_tma != 0, g, P, F, J, sc, ctx->d_counters,
                                                           ss.items, ss.d_n_items, ss.max_items, false,
                                                           ctx->tiled_attr[1][0], st, terr)
          : launch_step_tiled<real, Coord<real>, false>(ctx->tma, ctx->use_tma != 0, g, P, F, J, sc, ctx->d_counters,
                                                        ss.items, ss.d_n_items, ss.max_items, false,
                                                        ctx->tiled_attr[0][0], st, terr);
      if (!ok) return fail(ctx, GRPIC_ECUDA, terr);
      if (general_map(ctx))
        k_push_or_step_from<real, false, CoordGen<real>><<<kTailGrid, kBlock, 0, st>>>(g, P, F, J, sc, ctx->d_counters,
                                                                                       ss.d_n_items + 1);
      else
        k_push_or_step_from<real, false><<<kTailGrid, kBlock, 0, st>>>(g, P, F, J, sc, ctx->d_counters, ss.d_n_items + 1);
      CK(cudaGetLastError());
      return GRPIC_OK;
    }
  }
  if (general_map(ctx))
    k_push_or_step<real, false, CoordGen<real>><<<grid_for(p->n), kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), F, J, sc,
                                                                                   ctx->d_counters);
  else
    k_push_or_step<real, false><<<grid_for(p->n), kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), F, J, sc,
                                                                   ctx->d_counters);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_deposit(grpic_ctx* ctx, const grpic_particles* p, grpic_current* J, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, p, 1);
  if (rc) return rc;
  if (!ctx->have_dt) return fail(ctx, GRPIC_ESTATE, "grpic_deposit before any grpic_interp_push on this context");
  const SpeciesConst sc = make_species(p, ctx->last_dt, true);
  JPtrs<real> Jp;
  if ((rc = check_current(ctx, J, sc, Jp))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  CK(cudaMemsetAsync(ctx->d_counters + 3, 0, sizeof(unsigned long long), st));
  if (p->n == 0 || !sc.do_deposit) return GRPIC_OK;
  auto it = ctx->sorted.find((const void*)p->i1);
  if (ctx->tile_path && it != ctx->sorted.end() && table_covers(ctx, it->second, p)) {
    // sorted species: per-warp shared J tiles and warp aggregation instead of one L2 reduction per contribution
    const SortState& ss = it->second;
    std::string terr;
    const bool ok = general_map(ctx)
        ? launch_deposit_tiled<real, CoordGen<real>>(make_consts(ctx), make_pptrs(p), Jp, sc, ctx->d_counters, ss.items,
                                                     ss.d_n_items, ss.max_items, ctx->dep_attr[1], st, terr)
        : launch_deposit_tiled<real>(make_consts(ctx), make_pptrs(p), Jp, sc, ctx->d_counters, ss.items, ss.d_n_items,
                                     ss.max_items, ctx->dep_attr[0], st, terr);
    if (!ok) return fail(ctx, GRPIC_ECUDA, terr);
    if (general_map(ctx))
      k_deposit_from<real, CoordGen<real>><<<kTailGrid, kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), Jp, sc,
                                                                         ctx->d_counters, ss.d_n_items + 1);
    else
      k_deposit_from<real><<<kTailGrid, kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), Jp, sc, ctx->d_counters,
                                                         ss.d_n_items + 1);
    CK(cudaGetLastError());
    return GRPIC_OK;
  }
  if (general_map(ctx))
    k_deposit<real, CoordGen<real>><<<grid_for(p->n), kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), Jp, sc, ctx->d_counters);
  else
    k_deposit<real><<<grid_for(p->n), kBlock, 0, st>>>(make_consts(ctx), make_pptrs(p), Jp, sc, ctx->d_counters);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_step(grpic_ctx* ctx, grpic_particles* p, const grpic_fields* fields, grpic_current* J, double dt,
               void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, p, 2);
  if (rc) return rc;
  if (!(dt > 0.0)) return fail(ctx, GRPIC_EINVAL, "dt must be > 0");
  const SpeciesConst sc = make_species(p, dt, true);
  FPtrs<real> F;
  JPtrs<real> Jp;
  if ((rc = check_fields(ctx, fields, sc, F))) return rc;
  if ((rc = check_current(ctx, J, sc, Jp))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  ctx->last_dt = dt; ctx->have_dt = true;
  CK(cudaMemsetAsync(ctx->d_counters, 0, 4 * sizeof(unsigned long long), st));
  if (p->n == 0) return GRPIC_OK;
  const Consts<real> g = make_consts(ctx);
  const PPtrs<real> P = make_pptrs(p);

  auto it = ctx->sorted.find((const void*)p->i1);
  const bool tiled = ctx->tile_path && it != ctx->sorted.end() && sc.em && sc.do_deposit &&
                     table_covers(ctx, it->second, p);
  const bool gen = general_map(ctx);             // full A.3 map (r0, h0): same kernels, general coordinate class
  if (!tiled) {
    if (gen)
      k_push_or_step<real, true, CoordGen<real>><<<grid_for(p->n), kBlock, 0, st>>>(g, P, F, Jp, sc, ctx->d_counters);
    else
      k_push_or_step<real, true><<<grid_for(p->n), kBlock, 0, st>>>(g, P, F, Jp, sc, ctx->d_counters);
    CK(cudaGetLastError());
    return GRPIC_OK;
  }
  const SortState& ss = it->second;
  std::string terr;
  // dense items -> k_step_lanes (one run of particles per lane, 128-bit column blocks: every column 16-byte
  // aligned, as include/grpic.h requires; anything else keeps all items in k_step_tiled)
  bool lanes = ctx->lanes_path && ss.max_dense > 0;
  {
    const void* cols[10] = {p->i1, p->i2, p->dx1, p->dx2, p->u1, p->u2, p->u3, p->phi, p->weight, p->tag};
    for (const void* c : cols)
      if ((uintptr_t)c & 15u) lanes = false;
  }
  // With the lanes kernel on, the small kernels (sparse items, slots behind the alive count) go to a side stream of the
  // context, forked from and joined back into the caller's stream with events: submitted after k_step_lanes and at
  // lower priority, their blocks fill the SMs that the last wave of k_step_lanes leaves idle instead of adding their
  // ~0.15 ms in front of it.  (No host synchronisation; the pattern is capturable in a CUDA graph.)
  cudaStream_t side = st;
  bool ok = true;
  if (lanes && ctx->overlap) {
    if (!ctx->side_ok) {
      int lo = 0, hi = 0;
      cudaDeviceGetStreamPriorityRange(&lo, &hi);
      if (cudaStreamCreateWithPriority(&ctx->side, cudaStreamNonBlocking, lo) == cudaSuccess &&
          cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
          cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) == cudaSuccess)
        ctx->side_ok = true;
      else
        cudaGetLastError();
    }
    if (ctx->side_ok) {
      side = ctx->side;
      CK(cudaEventRecord(ctx->ev_fork, st));                // after the counter reset above
      CK(cudaStreamWaitEvent(side, ctx->ev_fork, 0));
    }
  }
  if (lanes)
    ok = gen ? launch_step_lanes<real, CoordGen<real>>(ctx->tma, ctx->use_tma != 0, g, P, F, Jp, sc, ctx->d_counters,
                                                       ss.items, ss.dense_idx, ss.d_n_items + 2, ss.offsets,
                                                       ss.max_dense, ctx->lanes_attr[1], st, terr)
             : launch_step_lanes<real>(ctx->tma, ctx->use_tma != 0, g, P, F, Jp, sc, ctx->d_counters, ss.items,
                                       ss.dense_idx, ss.d_n_items + 2, ss.offsets, ss.max_dense, ctx->lanes_attr[0],
                                       st, terr);
  if (ok)
    ok = gen ? launch_step_tiled<real, CoordGen<real>>(ctx->tma, ctx->use_tma != 0, g, P, F, Jp, sc, ctx->d_counters,
                                                       ss.items, ss.d_n_items, ss.max_items, lanes,
                                                       ctx->tiled_attr[1][1], side, terr)
             : launch_step_tiled<real>(ctx->tma, ctx->use_tma != 0, g, P, F, Jp, sc, ctx->d_counters, ss.items,
                                       ss.d_n_items, ss.max_items, lanes, ctx->tiled_attr[0][1], side, terr);
  if (!ok) return fail(ctx, GRPIC_ECUDA, terr);
  // slots behind the alive count of the sort (dead then; revived or appended since): direct path
  if (gen)
    k_push_or_step_from<real, true, CoordGen<real>><<<kTailGrid, kBlock, 0, side>>>(g, P, F, Jp, sc, ctx->d_counters,
                                                                                    ss.d_n_items + 1);
  else
    k_push_or_step_from<real, true><<<kTailGrid, kBlock, 0, side>>>(g, P, F, Jp, sc, ctx->d_counters, ss.d_n_items + 1);
  CK(cudaGetLastError());
  if (side != st) {
    CK(cudaEventRecord(ctx->ev_join, side));
    CK(cudaStreamWaitEvent(st, ctx->ev_join, 0));
  }
  return GRPIC_OK;
}

namespace {
// Counting sort of the columns of `src` into the columns of `p`.  src == p: in place from the caller's view
// (every column is first copied to library scratch); src != p: the gather reads the caller's source columns
// directly, no snapshot.  The *_prev columns and phi are optional (same set on both sides).
int sort_impl(grpic_ctx* ctx, const grpic_particles* src, grpic_particles* p, cudaStream_t st) {
  int rc;
  const int64_t n = p->n;
  if (n == 0) return GRPIC_OK;
  const bool in_place = (src == p);
  const bool has_prev = src->i1_prev != nullptr;
  const SortGeom sg = sort_geom(ctx);
  const uint32_t n_tiles = (uint32_t)sg.nt1 * sg.nt2;
  // scratch (grown on demand; growing synchronises)
  const size_t col = ((size_t)n * sizeof(real) + 255) / 256 * 256;
  const size_t col4 = ((size_t)n * 4 + 255) / 256 * 256;
  const size_t col1 = ((size_t)n + 255) / 256 * 256;
  const size_t need = in_place ? 9 * col + 4 * col4 + col1 : 256;
  if (ctx->cap_particles < n) {
    CK(cudaStreamSynchronize(st));
    cudaFree(ctx->d_keys); cudaFree(ctx->d_dest);
    ctx->d_keys = ctx->d_dest = nullptr; ctx->cap_particles = 0;
    if (cudaMalloc(&ctx->d_keys, (size_t)n * 4) != cudaSuccess || cudaMalloc(&ctx->d_dest, (size_t)n * 4) != cudaSuccess) {
      cudaGetLastError();
      return fail(ctx, GRPIC_ENOMEM, "sort scratch (keys) allocation failed");
    }
    ctx->cap_particles = n;
  }
  if (ctx->scratch_bytes < need) {
    CK(cudaStreamSynchronize(st));
    cudaFree(ctx->d_scratch); ctx->d_scratch = nullptr; ctx->scratch_bytes = 0;
    if (cudaMalloc(&ctx->d_scratch, need) != cudaSuccess) {
      cudaGetLastError();
      return fail(ctx, GRPIC_ENOMEM, "sort scratch (columns) allocation failed");
    }
    ctx->scratch_bytes = need;
  }
  if (!ctx->d_hist) {
    const uint32_t nb = (sg.n_keys + 1 + kScanTile - 1) / kScanTile + 1;
    if (cudaMalloc(&ctx->d_hist, ((size_t)sg.n_keys + 1) * 4) != cudaSuccess ||
        cudaMalloc(&ctx->d_block_sums, (size_t)(nb + 1024) * 4) != cudaSuccess ||
        cudaMalloc(&ctx->d_tile_items, ((size_t)n_tiles + 1) * 4) != cudaSuccess) {
      cudaGetLastError();
      return fail(ctx, GRPIC_ENOMEM, "sort scratch (histogram) allocation failed");
    }
  }
  // 1. keys + histogram; 2. exclusive scan -> offsets; 3. ranks (inverse permutation); 4. snapshot; 5. gather
  CK(cudaMemsetAsync(ctx->d_hist, 0, ((size_t)sg.n_keys + 1) * 4, st));
  SortPredict sp;
  {
    const FieldGeom q = make_field_geom(ctx);
    sp.on = (ctx->sort_lookahead > 0.0 && ctx->have_dt) ? 1 : 0;
    sp.tau = sp.on ? (float)(ctx->sort_lookahead * ctx->last_dt) : 0.0f;
    sp.log_rmin = (float)q.log_rmin; sp.dxi = (float)q.dxi; sp.r_off = (float)q.r_off; sp.r_min = (float)q.r_min;
    sp.dr = (float)q.dr; sp.deta = (float)q.deta; sp.h0 = (float)q.h0; sp.a = (float)q.a; sp.mass = (float)q.mass;
    sp.eps = src->massive ? 1.0f : 0.0f; sp.r_lin = q.r_lin;
  }
  k_sort_hist<real><<<(unsigned)((n + kBlock * kSortV - 1) / (kBlock * kSortV)), kBlock, 0, st>>>(
      sg, sp, n, src->i1, src->i2, src->tag, src->dx1, src->dx2, src->u1, src->u2, src->u3, ctx->d_keys, ctx->d_hist);
  if ((rc = scan_exclusive(ctx, ctx->d_hist, sg.n_keys + 1, st))) return rc;

  // tile table from the offsets (before the cursor copy is consumed).  Tables are keyed by the address of the i1
  // column; a caller that keeps allocating new columns would grow the map without bound, so the table of the species
  // sorted longest ago is dropped beyond kMaxTables (its next grpic_step simply takes the direct path).
  constexpr size_t kMaxTables = 64;
  if (ctx->sorted.find((const void*)p->i1) == ctx->sorted.end() && ctx->sorted.size() >= kMaxTables) {
    auto oldest = ctx->sorted.begin();
    for (auto it = ctx->sorted.begin(); it != ctx->sorted.end(); ++it)
      if (it->second.stamp < oldest->second.stamp) oldest = it;
    CK(cudaStreamSynchronize(st));
    free_sort_state(oldest->second);                   // cudaFree waits for work that may still read the table
    ctx->sorted.erase(oldest);
  }
  SortState& ss = ctx->sorted[(const void*)p->i1];
  ss.stamp = ++ctx->stamp;
  const uint32_t max_items = n_tiles + (uint32_t)((n + kChunk - 1) / kChunk);
  if (ss.max_items < max_items) {
    CK(cudaStreamSynchronize(st));
    free_sort_state(ss);
    if (cudaMalloc(&ss.items, (size_t)max_items * sizeof(WorkItem)) != cudaSuccess ||
        cudaMalloc(&ss.dense_idx, (size_t)max_items * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&ss.offsets, ((size_t)sg.n_keys + 1) * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&ss.d_n_items, 4 * sizeof(uint32_t)) != cudaSuccess) {
      cudaGetLastError();
      ctx->sorted.erase((const void*)p->i1);
      return fail(ctx, GRPIC_ENOMEM, "tile table allocation failed");
    }
    ss.max_items = max_items;
  }
  ss.n_at_sort = n;
  // the offsets outlive this call (k_step_lanes reads them); d_hist is about to become the rank cursor
  CK(cudaMemcpyAsync(ss.offsets, ctx->d_hist, ((size_t)sg.n_keys + 1) * sizeof(uint32_t), cudaMemcpyDeviceToDevice, st));
  k_items_count<<<(n_tiles + 255) / 256, 256, 0, st>>>(ctx->d_hist, n_tiles, ctx->d_tile_items);
  if ((rc = scan_exclusive(ctx, ctx->d_tile_items, n_tiles, st))) return rc;
  const uint32_t dense_min = ctx->lanes_path ? (uint32_t)ctx->dense_min : 0u;
  ss.max_dense = dense_min ? (uint32_t)std::min<int64_t>(max_items, n / dense_min) : 0u;
  CK(cudaMemsetAsync(ss.d_n_items, 0, 4 * sizeof(uint32_t), st));
  k_items_fill<<<(n_tiles + 255) / 256, 256, 0, st>>>(ctx->d_hist, n_tiles, ctx->d_tile_items, ss.items,
                                                      ss.d_n_items, ss.dense_idx, dense_min);

  k_sort_rank<<<(unsigned)((n + kBlock * kSortV - 1) / (kBlock * kSortV)), kBlock, 0, st>>>(n, ctx->d_keys, ctx->d_hist, ctx->d_dest);

  // in place: snapshot of every column in library scratch (plain contiguous copies); then ONE gather into the
  // destination columns in sorted order
  PPtrs<real> out = make_pptrs(p), in = make_pptrs(src);
  if (in_place) {
    char* s = (char*)ctx->d_scratch;
    in.dx1 = (real*)s; s += col; in.dx2 = (real*)s; s += col;
    in.u1 = (real*)s; s += col; in.u2 = (real*)s; s += col; in.u3 = (real*)s; s += col;
    in.phi = p->phi ? (real*)s : nullptr; s += col;
    in.dx1p = has_prev ? (real*)s : nullptr; s += col; in.dx2p = has_prev ? (real*)s : nullptr; s += col;
    in.w = (const real*)s; s += col;
    in.i1 = (int32_t*)s; s += col4; in.i2 = (int32_t*)s; s += col4;
    in.i1p = has_prev ? (int32_t*)s : nullptr; s += col4; in.i2p = has_prev ? (int32_t*)s : nullptr; s += col4;
    in.tag = (uint8_t*)s;
    const size_t rb = (size_t)n * sizeof(real), ib = (size_t)n * 4;
    CK(cudaMemcpyAsync(in.dx1, p->dx1, rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.dx2, p->dx2, rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.u1, p->u1, rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.u2, p->u2, rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.u3, p->u3, rb, cudaMemcpyDeviceToDevice, st));
    if (p->phi) CK(cudaMemcpyAsync(in.phi, p->phi, rb, cudaMemcpyDeviceToDevice, st));
    if (has_prev) {
      CK(cudaMemcpyAsync(in.dx1p, p->dx1_prev, rb, cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(in.dx2p, p->dx2_prev, rb, cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(in.i1p, p->i1_prev, ib, cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(in.i2p, p->i2_prev, ib, cudaMemcpyDeviceToDevice, st));
    }
    CK(cudaMemcpyAsync((void*)in.w, p->weight, rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.i1, p->i1, ib, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.i2, p->i2, ib, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(in.tag, p->tag, (size_t)n, cudaMemcpyDeviceToDevice, st));
  }
  k_sort_gather<real><<<(unsigned)((n + kBlock * kGatherV - 1) / (kBlock * kGatherV)), kBlock, 0, st>>>(in, out, ctx->d_dest);
  CK(cudaGetLastError());
  // the number of alive particles (they now occupy [0, n_alive)) stays on the device: the kernels read it there
  ss.n_alive_known = false;
  ss.stream = st;
  return GRPIC_OK;
}
}  // namespace

int grpic_sort(grpic_ctx* ctx, grpic_particles* p, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, p, 2);
  if (rc) return rc;
  return sort_impl(ctx, p, p, (cudaStream_t)stream);
}

int grpic_sort_into(grpic_ctx* ctx, const grpic_particles* src, grpic_particles* dst, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, src, 2);
  if (rc || (rc = check_particles(ctx, dst, 2))) return rc;
  if (src->n != dst->n) return fail(ctx, GRPIC_EINVAL, "sort_into: src.n != dst.n");
  if (src->n == 0) return GRPIC_OK;
  if ((src->phi != nullptr) != (dst->phi != nullptr) || (src->i1_prev != nullptr) != (dst->i1_prev != nullptr))
    return fail(ctx, GRPIC_EINVAL, "sort_into: src and dst must carry the same optional columns");
  // no column of dst may be a column of src (the gather reads src while dst is written)
  const void* a[14] = {src->i1, src->i2, src->dx1, src->dx2, src->u1, src->u2, src->u3, src->phi, src->i1_prev,
                       src->i2_prev, src->dx1_prev, src->dx2_prev, src->weight, src->tag};
  const void* b[14] = {dst->i1, dst->i2, dst->dx1, dst->dx2, dst->u1, dst->u2, dst->u3, dst->phi, dst->i1_prev,
                       dst->i2_prev, dst->dx1_prev, dst->dx2_prev, dst->weight, dst->tag};
  for (int i = 0; i < 14; ++i)
    for (int j = 0; j < 14; ++j)
      if (a[i] && a[i] == b[j]) return fail(ctx, GRPIC_EINVAL, "sort_into: src and dst share a column");
  return sort_impl(ctx, src, dst, (cudaStream_t)stream);
}

int grpic_forget(grpic_ctx* ctx, const grpic_particles* p) {
  if (!ctx || !p) return fail(ctx, GRPIC_EINVAL, "NULL argument");
  auto it = ctx->sorted.find((const void*)p->i1);
  if (it == ctx->sorted.end()) return GRPIC_OK;
  if (int rd = check_device(ctx)) return rd;
  free_sort_state(it->second);                         // cudaFree waits for work that may still read the table
  ctx->sorted.erase(it);
  return GRPIC_OK;
}

int grpic_sorted_alive(grpic_ctx* ctx, const grpic_particles* p, int64_t* n_alive) {
  if (!ctx || !p || !n_alive) return fail(ctx, GRPIC_EINVAL, "NULL argument");
  auto it = ctx->sorted.find((const void*)p->i1);
  if (it == ctx->sorted.end()) return fail(ctx, GRPIC_ESTATE, "this species has not been sorted on this context");
  int rc = fetch_alive(ctx, it->second);
  if (rc) return rc;
  *n_alive = it->second.n_alive;
  return GRPIC_OK;
}

int grpic_counters(grpic_ctx* ctx, int64_t* n_alive, int64_t* n_in, int64_t* n_out, int64_t* n_over, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  unsigned long long h[4];
  CK(cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CK(cudaStreamSynchronize((cudaStream_t)stream));
  if (n_alive) *n_alive = (int64_t)h[0];
  if (n_in) *n_in = (int64_t)h[1];
  if (n_out) *n_out = (int64_t)h[2];
  if (n_over) *n_over = (int64_t)h[3];
  return GRPIC_OK;
}

int grpic_probe(grpic_ctx* ctx, const char* what, int64_t iters, int64_t* ops, void* stream) {
  if (!ctx || !what || !ops) return fail(ctx, GRPIC_EINVAL, "NULL argument");
  if (int rd = check_device(ctx)) return rd;
  if (iters < 1 || iters > (1 << 24)) return fail(ctx, GRPIC_EINVAL, "iters must be in 1..2^24");
  cudaStream_t st = (cudaStream_t)stream;
  const int grid = 148 * 8;
  float* out = reinterpret_cast<float*>(ctx->d_counters + 6);            // a spare word, never written in practice
  const int64_t lane_ops = (int64_t)grid * kProbeBlock * kProbeChains * 8 * iters;
  if (!std::strcmp(what, "ffma")) { k_probe<0><<<grid, kProbeBlock, 0, st>>>((int)iters, 1.0f, out); *ops = 2 * lane_ops; }
  else if (!std::strcmp(what, "dfma")) { k_probe<1><<<grid, kProbeBlock, 0, st>>>((int)iters, 1.0f, out); *ops = 2 * lane_ops; }
  else if (!std::strcmp(what, "mufu")) { k_probe<2><<<grid, kProbeBlock, 0, st>>>((int)iters, 1.0f, out); *ops = lane_ops; }
  else if (!std::strcmp(what, "smem_rmw")) { k_probe<3><<<grid, kProbeBlock, 0, st>>>((int)iters, 1.0f, out); *ops = lane_ops; }
  else return fail(ctx, GRPIC_EINVAL, std::string("unknown probe: ") + what);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_updates_total(grpic_ctx* ctx, int64_t* n_updates, void* stream) {
  if (!ctx || !n_updates) return fail(ctx, GRPIC_EINVAL, "ctx or n_updates is NULL");
  unsigned long long h = 0;
  CK(cudaMemcpyAsync(&h, ctx->d_counters + 4, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CK(cudaStreamSynchronize((cudaStream_t)stream));
  *n_updates = (int64_t)h;
  return GRPIC_OK;
}

// ------------------------------------------------------------------------------------------------
// Field-solver half: auxiliary fields, Faraday, Ampere
// ------------------------------------------------------------------------------------------------
int grpic_aux_fields(grpic_ctx* ctx, const grpic_fields* em, grpic_vec3* E, grpic_vec3* H, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!em || !em->D1 || !em->D2 || !em->D3 || !em->B1 || !em->B2 || !em->B3)
    return fail(ctx, GRPIC_EINVAL, "a field component pointer is NULL");
  if (!E && !H) return fail(ctx, GRPIC_EINVAL, "both outputs are NULL");
  if ((E && (!E->F1 || !E->F2 || !E->F3)) || (H && (!H->F1 || !H->F2 || !H->F3)))
    return fail(ctx, GRPIC_EINVAL, "an output component pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  FPtrs<real> F;
  F.f[0] = em->D1; F.f[1] = em->D2; F.f[2] = em->D3; F.f[3] = em->B1; F.f[4] = em->B2; F.f[5] = em->B3;
  V3<real> Ev{{E ? E->F1 : nullptr, E ? E->F2 : nullptr, E ? E->F3 : nullptr}};
  V3<real> Hv{{H ? H->F1 : nullptr, H ? H->F2 : nullptr, H ? H->F3 : nullptr}};
  const dim3 grid((q.n2 + 1 + 127) / 128, q.rows - 2);
  k_aux_fields<real><<<grid, 128, 0, (cudaStream_t)stream>>>(q, F, Ev, Hv);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_faraday(grpic_ctx* ctx, grpic_vec3* B, const grpic_vec3* E, double dt, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!B || !E || !B->F1 || !B->F2 || !B->F3 || !E->F1 || !E->F2 || !E->F3)
    return fail(ctx, GRPIC_EINVAL, "a component pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  if (q.rows < 5) return GRPIC_OK;
  V3<real> Bv{{B->F1, B->F2, B->F3}};
  CV3<real> Ev{{E->F1, E->F2, E->F3}};
  const dim3 grid((q.n2 + 127) / 128, q.rows - 4);
  k_faraday<real><<<grid, 128, 0, (cudaStream_t)stream>>>(q, Bv, Ev, dt);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_ampere(grpic_ctx* ctx, grpic_vec3* D, const grpic_vec3* H, const grpic_current* J, double dt, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!D || !H || !D->F1 || !D->F2 || !D->F3 || !H->F1 || !H->F2 || !H->F3)
    return fail(ctx, GRPIC_EINVAL, "a component pointer is NULL");
  if (J && (!J->J1 || !J->J2 || !J->J3)) return fail(ctx, GRPIC_EINVAL, "a current component pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  if (q.rows < 5) return GRPIC_OK;
  V3<real> Dv{{D->F1, D->F2, D->F3}};
  CV3<real> Hv{{H->F1, H->F2, H->F3}};
  CV3<real> Jv{{J ? J->J1 : nullptr, J ? J->J2 : nullptr, J ? J->J3 : nullptr}};
  const dim3 grid((q.n2 + 1 + 127) / 128, q.rows - 4);
  k_ampere<real><<<grid, 128, 0, (cudaStream_t)stream>>>(q, Dv, Hv, Jv, ctx->k_J, dt);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_field_bc(grpic_ctx* ctx, grpic_vec3* D, grpic_vec3* B, int32_t n_const, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!D || !B || !D->F1 || !D->F2 || !D->F3 || !B->F1 || !B->F2 || !B->F3)
    return fail(ctx, GRPIC_EINVAL, "a component pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  if (n_const >= q.n1) return fail(ctx, GRPIC_EINVAL, "n_const must be < n1");
  if (q.n2 < q.ng) return fail(ctx, GRPIC_EINVAL, "n2 must be >= nghost for the axis reflection");
  V3<real> Dv{{D->F1, D->F2, D->F3}}, Bv{{B->F1, B->F2, B->F3}};
  cudaStream_t st = (cudaStream_t)stream;
  k_field_bc_axis<real><<<dim3(1, q.rows, 6), 128, 0, st>>>(q, Dv, Bv, 0);
  if (n_const >= 0)
    k_field_bc_layer<real><<<dim3((q.ld + 127) / 128, q.ng + n_const + 1, 6), 128, 0, st>>>(q, Dv, Bv, n_const);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_field_match(grpic_ctx* ctx, grpic_vec3* D, grpic_vec3* B, const grpic_vec3* D_target, const grpic_vec3* B_target,
                      double r_abs, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!D || !B || !D->F1 || !D->F2 || !D->F3 || !B->F1 || !B->F2 || !B->F3 || !D_target || !B_target ||
      !D_target->F1 || !D_target->F2 || !D_target->F3 || !B_target->F1 || !B_target->F2 || !B_target->F3)
    return fail(ctx, GRPIC_EINVAL, "a component pointer is NULL");
  if (!(r_abs >= ctx->r_min && r_abs < ctx->r_max)) return fail(ctx, GRPIC_EINVAL, "r_abs must be in [r_min, r_max)");
  const FieldGeom q = make_field_geom(ctx);
  // first array row that can lie in the layer: the cell that holds r_abs
  double x1;
  if (q.r_lin) x1 = (r_abs - q.r_min) / q.dr;
  else x1 = (std::log(r_abs - q.r_off) - q.log_rmin) / q.dxi;
  int row0 = (int)std::floor(x1) - 1 + q.ng;
  if (row0 < 0) row0 = 0;
  V3<real> Dv{{D->F1, D->F2, D->F3}}, Bv{{B->F1, B->F2, B->F3}};
  CV3<real> D0{{D_target->F1, D_target->F2, D_target->F3}}, B0{{B_target->F1, B_target->F2, B_target->F3}};
  k_field_match<real><<<dim3((q.ld + 127) / 128, q.rows - row0, 6), 128, 0, (cudaStream_t)stream>>>(
      q, Dv, Bv, D0, B0, r_abs, ctx->r_max, row0);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

// ---- field side of one PIC timestep (Sec. 3.4) ----
namespace {
int field_scratch(grpic_ctx* ctx, size_t cells) {
  if (ctx->f_scratch_cells >= cells) return GRPIC_OK;
  cudaFree(ctx->f_scratch); ctx->f_scratch = nullptr; ctx->f_scratch_cells = 0;
  if (cudaMalloc((void**)&ctx->f_scratch, 12 * cells * sizeof(real)) != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, GRPIC_ENOMEM, "field scratch allocation failed");
  }
  ctx->f_scratch_cells = cells;
  return GRPIC_OK;
}
bool vec3_ok(const grpic_vec3* v) { return v && v->F1 && v->F2 && v->F3; }
void average3(real* out, const real* a1, const real* a2, const real* a3, const real* b1, const real* b2, const real* b3,
              size_t cells, cudaStream_t st) {
  const unsigned nb = (unsigned)((cells + 255) / 256);
  k_average<real><<<nb, 256, 0, st>>>(out, a1, b1, (int64_t)cells);
  k_average<real><<<nb, 256, 0, st>>>(out + cells, a2, b2, (int64_t)cells);
  k_average<real><<<nb, 256, 0, st>>>(out + 2 * cells, a3, b3, (int64_t)cells);
}
}  // namespace

int grpic_filter_current(grpic_ctx* ctx, grpic_current* J, int32_t n_passes, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!J || !J->J1 || !J->J2 || !J->J3) return fail(ctx, GRPIC_EINVAL, "a current component pointer is NULL");
  if (n_passes < 0) return fail(ctx, GRPIC_EINVAL, "n_passes must be >= 0");
  const FieldGeom q = make_field_geom(ctx);
  if (q.n2 < 2) return fail(ctx, GRPIC_EINVAL, "n2 must be >= 2 for the filter");
  const size_t cells = (size_t)q.rows * q.ld, bytes = cells * sizeof(real);
  int rc = field_scratch(ctx, cells);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  real* S = ctx->f_scratch;
  real* Jp[3] = {J->J1, J->J2, J->J3};
  for (int pass = 0; pass < n_passes; ++pass) {
    // scratch <- J (ghost columns and all), then J <- filter(scratch) on the physical samples
    for (int c = 0; c < 3; ++c) CK(cudaMemcpyAsync(S + c * cells, Jp[c], bytes, cudaMemcpyDeviceToDevice, st));
    CV3<real> in{{S, S + cells, S + 2 * cells}};
    V3<real> out{{Jp[0], Jp[1], Jp[2]}};
    k_filter_current<real><<<dim3((q.n2 + 1 + 127) / 128, q.rows, 3), 128, 0, st>>>(q, in, out);
  }
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_fields_prepare(grpic_ctx* ctx, const grpic_field_state* s, grpic_vec3* B_n, double dt, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!s || !vec3_ok(&s->B_prev) || !vec3_ok(&s->B) || !vec3_ok(&s->D_prev) || !vec3_ok(&s->D) || !vec3_ok(B_n))
    return fail(ctx, GRPIC_EINVAL, "a field pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  const size_t cells = (size_t)q.rows * q.ld;
  int rc = field_scratch(ctx, cells);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  real* E = ctx->f_scratch; real* Dh = ctx->f_scratch + 6 * cells;
  const unsigned nb = (unsigned)((cells + 255) / 256);
  // Eq. 46: (n-1)B = ((n-3/2)B + (n-1/2)B)/2 -> B_n;  (n-1/2)D = ((n-1)D + (n)D)/2
  k_average<real><<<nb, 256, 0, st>>>(B_n->F1, s->B_prev.F1, s->B.F1, (int64_t)cells);
  k_average<real><<<nb, 256, 0, st>>>(B_n->F2, s->B_prev.F2, s->B.F2, (int64_t)cells);
  k_average<real><<<nb, 256, 0, st>>>(B_n->F3, s->B_prev.F3, s->B.F3, (int64_t)cells);
  average3(Dh, s->D_prev.F1, s->D_prev.F2, s->D_prev.F3, s->D.F1, s->D.F2, s->D.F3, cells, st);
  // Eq. 47: (n-1/2)E from (n-1/2)B, (n-1/2)D
  FPtrs<real> F;
  F.f[0] = Dh; F.f[1] = Dh + cells; F.f[2] = Dh + 2 * cells; F.f[3] = s->B.F1; F.f[4] = s->B.F2; F.f[5] = s->B.F3;
  V3<real> Ev{{E, E + cells, E + 2 * cells}}, none{{nullptr, nullptr, nullptr}};
  k_aux_fields<real><<<dim3((q.n2 + 1 + 127) / 128, q.rows - 2), 128, 0, st>>>(q, F, Ev, none);
  // Eq. 48: (n-1)B -> (n)B
  if (q.rows >= 5) {
    V3<real> Bv{{B_n->F1, B_n->F2, B_n->F3}};
    CV3<real> Ec{{E, E + cells, E + 2 * cells}};
    k_faraday<real><<<dim3((q.n2 + 127) / 128, q.rows - 4), 128, 0, st>>>(q, Bv, Ec, dt);
  }
  // (n)B is what the particle gather reads, ghost columns beyond the axes included (node averages of B^1, B^3 in
  // the cells next to an axis): Faraday wrote the physical columns only, so the axis reflection is applied
  // to (n)B here - otherwise its ghost columns would still hold the time level n-1
  if (q.n2 >= q.ng) {
    V3<real> Bv{{B_n->F1, B_n->F2, B_n->F3}};
    k_field_bc_axis<real><<<dim3(1, q.rows, 3), 128, 0, st>>>(q, Bv, Bv, 3);
  }
  CK(cudaGetLastError());
  return GRPIC_OK;
}

int grpic_fields_advance(grpic_ctx* ctx, grpic_field_state* s, const grpic_vec3* B_n, const grpic_current* J_prev,
                         const grpic_current* J, double dt, void* stream) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  if (!s || !vec3_ok(&s->B_prev) || !vec3_ok(&s->B) || !vec3_ok(&s->D_prev) || !vec3_ok(&s->D) || !vec3_ok(B_n))
    return fail(ctx, GRPIC_EINVAL, "a field pointer is NULL");
  if ((J == nullptr) != (J_prev == nullptr)) return fail(ctx, GRPIC_EINVAL, "J and J_prev must both be given or both be NULL");
  if (J && (!J->J1 || !J->J2 || !J->J3 || !J_prev->J1 || !J_prev->J2 || !J_prev->J3))
    return fail(ctx, GRPIC_EINVAL, "a current component pointer is NULL");
  const FieldGeom q = make_field_geom(ctx);
  const size_t cells = (size_t)q.rows * q.ld, bytes = cells * sizeof(real);
  int rc = field_scratch(ctx, cells);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  real *E = ctx->f_scratch, *H = E + 3 * cells, *Dh = E + 6 * cells, *Jn = E + 9 * cells;
  const dim3 g_aux((q.n2 + 1 + 127) / 128, q.rows - 2), g_far((q.n2 + 127) / 128, q.rows - 4), g_amp((q.n2 + 1 + 127) / 128, q.rows - 4);
  V3<real> Ev{{E, E + cells, E + 2 * cells}}, Hv{{H, H + cells, H + 2 * cells}}, none{{nullptr, nullptr, nullptr}};
  CV3<real> Ec{{E, E + cells, E + 2 * cells}}, Hc{{H, H + cells, H + 2 * cells}};
  // Eq. 51: (n)J = ((n-1/2)J + (n+1/2)J)/2
  CV3<real> Jnc{{nullptr, nullptr, nullptr}}, Jc{{nullptr, nullptr, nullptr}};
  if (J) {
    average3(Jn, J_prev->J1, J_prev->J2, J_prev->J3, J->J1, J->J2, J->J3, cells, st);
    Jnc = CV3<real>{{Jn, Jn + cells, Jn + 2 * cells}};
    Jc = CV3<real>{{J->J1, J->J2, J->J3}};
  }
  // Eq. 52: (n)E, (n)H from (n)B, (n)D
  FPtrs<real> F;
  F.f[0] = s->D.F1; F.f[1] = s->D.F2; F.f[2] = s->D.F3; F.f[3] = B_n->F1; F.f[4] = B_n->F2; F.f[5] = B_n->F3;
  k_aux_fields<real><<<g_aux, 128, 0, st>>>(q, F, Ev, Hv);
  // (n-1/2)D before D is touched
  average3(Dh, s->D_prev.F1, s->D_prev.F2, s->D_prev.F3, s->D.F1, s->D.F2, s->D.F3, cells, st);
  // Eq. 53: (n-1/2)B -> (n+1/2)B; the old (n-1/2)B moves to B_prev
  CK(cudaMemcpyAsync(s->B_prev.F1, s->B.F1, bytes, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(s->B_prev.F2, s->B.F2, bytes, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(s->B_prev.F3, s->B.F3, bytes, cudaMemcpyDeviceToDevice, st));
  if (q.rows >= 5) k_faraday<real><<<g_far, 128, 0, st>>>(q, V3<real>{{s->B.F1, s->B.F2, s->B.F3}}, Ec, dt);
  // Eq. 54: (n-1/2)D -> (n+1/2)D with (n)H, (n)J
  if (q.rows >= 5) k_ampere<real><<<g_amp, 128, 0, st>>>(q, V3<real>{{Dh, Dh + cells, Dh + 2 * cells}}, Hc, Jnc, ctx->k_J, dt);
  // Eq. 55: (n+1/2)H from (n+1/2)B, (n+1/2)D
  F.f[0] = Dh; F.f[1] = Dh + cells; F.f[2] = Dh + 2 * cells; F.f[3] = s->B.F1; F.f[4] = s->B.F2; F.f[5] = s->B.F3;
  k_aux_fields<real><<<g_aux, 128, 0, st>>>(q, F, none, Hv);
  // Eq. 56: (n)D -> (n+1)D with (n+1/2)H, (n+1/2)J; the old (n)D moves to D_prev
  CK(cudaMemcpyAsync(s->D_prev.F1, s->D.F1, bytes, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(s->D_prev.F2, s->D.F2, bytes, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(s->D_prev.F3, s->D.F3, bytes, cudaMemcpyDeviceToDevice, st));
  if (q.rows >= 5) k_ampere<real><<<g_amp, 128, 0, st>>>(q, V3<real>{{s->D.F1, s->D.F2, s->D.F3}}, Hc, Jc, ctx->k_J, dt);
  CK(cudaGetLastError());
  return GRPIC_OK;
}

// ------------------------------------------------------------------------------------------------
// Host-buffer end-to-end step: chunked H2D -> fused step -> D2H on two streams.
// ------------------------------------------------------------------------------------------------
int grpic_step_host(grpic_ctx* ctx, grpic_particles* ph, const grpic_fields* fh, grpic_current* Jh, double dt,
                    int64_t* h2d_bytes, int64_t* d2h_bytes) {
  if (!ctx) return GRPIC_EINVAL;
  if (int rd = check_device(ctx)) return rd;
  int rc = check_particles(ctx, ph, 0);
  if (rc) return rc;
  const bool want_prev = ph->i1_prev && ph->i2_prev && ph->dx1_prev && ph->dx2_prev;   // all four or none come back
  if (!(dt > 0.0)) return fail(ctx, GRPIC_EINVAL, "dt must be > 0");
  const SpeciesConst sc = make_species(ph, dt, true);
  if (sc.em && (!fh || !fh->D1 || !fh->D2 || !fh->D3 || !fh->B1 || !fh->B2 || !fh->B3))
    return fail(ctx, GRPIC_EINVAL, "host field pointers are NULL for a charged massive species");
  if (sc.do_deposit && (!Jh || !Jh->J1 || !Jh->J2 || !Jh->J3))
    return fail(ctx, GRPIC_EINVAL, "host current pointers are NULL for a charged species");
  int64_t up = 0, down = 0;
  const size_t cells = (size_t)(ctx->grid.n1 + 2 * ctx->grid.nghost) * (ctx->grid.n2 + 2 * ctx->grid.nghost);
  const size_t gbytes = cells * sizeof(real);
  if (!ctx->h_streams_ok) {
    for (auto& q : ctx->h_streams) CK(cudaStreamCreateWithFlags(&q, cudaStreamNonBlocking));
    ctx->h_streams_ok = true;
  }
  if (ctx->h_fields_bytes < 9 * gbytes) {
    cudaFree(ctx->h_fields); ctx->h_fields = nullptr; ctx->h_fields_bytes = 0;
    if (cudaMalloc(&ctx->h_fields, 9 * gbytes) != cudaSuccess) {
      cudaGetLastError();
      return fail(ctx, GRPIC_ENOMEM, "device grid buffers allocation failed");
    }
    ctx->h_fields_bytes = 9 * gbytes;
  }
  // particles per chunk: three chunks in flight.  Measured on config 4 (ms per step, both species): 2^22 117.5,
  // 2^21 118.6, 2^20 125.5, 2^18 170 - below 4 MB per column copy the per-copy cost of the engines shows
  const int64_t chunk = ctx->host_chunk;
  const size_t cb = (size_t)chunk * 8;                 // widest column
  if (ctx->h_cap < cb) {
    for (auto& q : ctx->h_dev) { cudaFree(q); q = nullptr; }
    ctx->h_cap = 0;
    for (auto& q : ctx->h_dev)
      if (cudaMalloc(&q, 3 * cb) != cudaSuccess) {      // three chunks in flight: upload, compute, download
        cudaGetLastError();
        return fail(ctx, GRPIC_ENOMEM, "device particle chunk allocation failed");
      }
    ctx->h_cap = cb;
  }
  cudaStream_t s0 = ctx->h_streams[0];
  real* dgrid = (real*)ctx->h_fields;
  FPtrs<real> F;
  for (int k = 0; k < 6; ++k) F.f[k] = nullptr;
  if (sc.em) {
    const real* src[6] = {fh->D1, fh->D2, fh->D3, fh->B1, fh->B2, fh->B3};
    for (int k = 0; k < 6; ++k) {
      CK(cudaMemcpyAsync(dgrid + k * cells, src[k], gbytes, cudaMemcpyHostToDevice, s0));
      F.f[k] = dgrid + k * cells;
      up += (int64_t)gbytes;
    }
  }
  JPtrs<real> Jp{{nullptr, nullptr, nullptr}};
  if (sc.do_deposit) {
    // J_host += : the host values go up, the deposit adds on the device, the sums come back
    real* src[3] = {Jh->J1, Jh->J2, Jh->J3};
    for (int k = 0; k < 3; ++k) {
      Jp.j[k] = dgrid + (6 + k) * cells;
      CK(cudaMemcpyAsync(Jp.j[k], src[k], gbytes, cudaMemcpyHostToDevice, s0));
      up += (int64_t)gbytes;
    }
  }
  CK(cudaMemsetAsync(ctx->d_counters, 0, 4 * sizeof(unsigned long long), s0));
  CK(cudaStreamSynchronize(s0));
  ctx->last_dt = dt; ctx->have_dt = true;
  const Consts<real> g = make_consts(ctx);
  // chunk sizes: the first upload and the last download of a call overlap nothing, so a long call ramps up
  // (chunk/8, /4, /2), runs full chunks, and ramps down again
  std::vector<int64_t> sizes;
  {
    int64_t body = ph->n;
    const int64_t ramp[3] = {chunk / 8, chunk / 4, chunk / 2};
    const bool ramped = ph->n >= 4 * chunk && chunk >= 8192;
    if (ramped) {
      for (int k = 0; k < 3; ++k) { sizes.push_back(ramp[k]); body -= 2 * ramp[k]; }
    }
    for (; body > 0; body -= chunk) sizes.push_back(body < chunk ? body : chunk);
    if (ramped)
      for (int k = 2; k >= 0; --k) sizes.push_back(ramp[k]);
  }
  int buf = 0;
  int64_t lo = 0;
  for (size_t ci = 0; ci < sizes.size(); lo += sizes[ci], ++ci, buf = (buf + 1) % 3) {
    const int64_t m = sizes[ci];
    cudaStream_t st = ctx->h_streams[buf];
    char* base[16];
    for (int k = 0; k < 16; ++k) base[k] = (char*)ctx->h_dev[k] + (size_t)buf * cb;
    PPtrs<real> P;
    P.n = m;
    P.i1 = (int32_t*)base[0]; P.i2 = (int32_t*)base[1];
    P.dx1 = (real*)base[2]; P.dx2 = (real*)base[3];
    P.u1 = (real*)base[4]; P.u2 = (real*)base[5]; P.u3 = (real*)base[6];
    P.phi = ph->phi ? (real*)base[7] : nullptr;
    P.i1p = want_prev ? (int32_t*)base[8] : nullptr; P.i2p = want_prev ? (int32_t*)base[9] : nullptr;
    P.dx1p = want_prev ? (real*)base[10] : nullptr; P.dx2p = want_prev ? (real*)base[11] : nullptr;
    P.w = (const real*)base[12]; P.tag = (uint8_t*)base[13];
    const size_t rb = (size_t)m * sizeof(real), ib = (size_t)m * 4;
#define UP(dst, src, bytes) do { CK(cudaMemcpyAsync((void*)(dst), (src) + lo, bytes, cudaMemcpyHostToDevice, st)); up += (int64_t)(bytes); } while (0)
#define DOWN(dst, src, bytes) do { CK(cudaMemcpyAsync((dst) + lo, (src), bytes, cudaMemcpyDeviceToHost, st)); down += (int64_t)(bytes); } while (0)
    UP(P.i1, ph->i1, ib); UP(P.i2, ph->i2, ib);
    UP(P.dx1, ph->dx1, rb); UP(P.dx2, ph->dx2, rb);
    UP(P.u1, ph->u1, rb); UP(P.u2, ph->u2, rb); UP(P.u3, ph->u3, rb);
    if (P.phi) UP(P.phi, ph->phi, rb);
    UP(P.w, ph->weight, rb); UP(P.tag, ph->tag, (size_t)m);
    if (general_map(ctx))
      k_push_or_step<real, true, CoordGen<real>><<<grid_for(m), kBlock, 0, st>>>(g, P, F, Jp, sc, ctx->d_counters);
    else
      k_push_or_step<real, true><<<grid_for(m), kBlock, 0, st>>>(g, P, F, Jp, sc, ctx->d_counters);
    CK(cudaGetLastError());
    DOWN(ph->i1, P.i1, ib); DOWN(ph->i2, P.i2, ib);
    DOWN(ph->dx1, P.dx1, rb); DOWN(ph->dx2, P.dx2, rb);
    DOWN(ph->u1, P.u1, rb); DOWN(ph->u2, P.u2, rb); DOWN(ph->u3, P.u3, rb);
    if (P.phi) DOWN(ph->phi, P.phi, rb);
    if (want_prev) {
      DOWN(ph->i1_prev, P.i1p, ib); DOWN(ph->i2_prev, P.i2p, ib);
      DOWN(ph->dx1_prev, P.dx1p, rb); DOWN(ph->dx2_prev, P.dx2p, rb);
    }
    DOWN(ph->tag, P.tag, (size_t)m);
#undef UP
#undef DOWN
  }
  for (auto& q : ctx->h_streams) CK(cudaStreamSynchronize(q));
  if (sc.do_deposit) {
    real* dst[3] = {Jh->J1, Jh->J2, Jh->J3};
    for (int k = 0; k < 3; ++k) {
      CK(cudaMemcpyAsync(dst[k], Jp.j[k], gbytes, cudaMemcpyDeviceToHost, s0));
      down += (int64_t)gbytes;
    }
    CK(cudaStreamSynchronize(s0));
  }
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return GRPIC_OK;
}

}  // extern "C"
