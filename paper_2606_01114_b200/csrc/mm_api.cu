// C ABI of include/mm_b200.h: context, workspace carve-up, call sequencing.  Every numeric
// step runs in the kernels of demag_passes.cu / demag_init.cu / pointwise.cu; this file only
// validates arguments and enqueues launches on the context's stream.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/mm_b200.h"
#include "bb.cuh"
#include "demag_fast.cuh"
#include "demag_init.cuh"
#include "demag_mixed.cuh"
#include "demag_passes.cuh"
#include "demag_ztile.cuh"
#include "fft_core.cuh"
#include "pointwise.cuh"
#include "rkf45.cuh"

using namespace mm;

static const double kMu0 = 4.0e-7 * 3.14159265358979323846;  // reading Q8
static char g_create_error[256] = "";

struct mm_ctx {
  int nx, ny, nz;
  double dx, dy, dz;
  mm_dtype dtype;
  size_t es;  // bytes per real
  cudaStream_t stream = nullptr;
  // material / terms
  bool have_material = false;
  double Ms = 0, Aex = 0, Ku = 0, axis[3] = {0, 0, 1}, alpha = 0, gamma = 2.211e5;
  double Hext[3] = {0, 0, 0};
  double Ddmi = 0, edmi[9] = {0, 1, 0, -1, 0, 0, 0, 0, 0};   // interfacial vectors by default
  double stt_p[3] = {0, 0, 1}, stt_damp = 0, stt_field = 0;
  const void* ms_cells = nullptr;   // per-cell Ms / A (device, ctx dtype, caller-owned), or NULL = uniform
  const void* a_cells = nullptr;
  unsigned terms = MM_TERM_DEMAG | MM_TERM_EXCHANGE;
  // plan
  DemagGeom geom{};
  InitGeom igeom{};
  FastGeom fgeom{};
  bool fast = false;     // the x-first kernels of demag_fast.cu cover this mesh and are selected
  bool mixed = false;    // the mixed-radix x-first kernels of demag_mixed.cu are selected
  bool embed = false;    // the demag passes run on the enclosing power-of-two mesh dnx x dny x dnz
  int dnx = 0, dny = 0, dnz = 0;   // mesh of the demag passes (= nx, ny, nz unless embedded)
  int nzt = 0;                      // x-first path: the z transform has period 2 nzt >= 2 dnz (demag_fast.cuh)
  int slabs = 0;                    // > 0: slab decomposition over this many (emulated) ranks, demag_fast.cuh SlabView
  int slab_rpr() const { return (dny + 1 + slabs - 1) / slabs; }   // ky rows per rank
  bool xfirst() const { return fast || mixed; }   // x-first spectra and the octant table
  int path_pref = 0;     // 0 auto, 1 generic (demag_passes.cu), 2 fast required
  int want_bz = 0, want_by = 0, want_bk = 0;
  // workspaces
  unsigned char* pers = nullptr;
  unsigned char* scr = nullptr;
  size_t pers_bytes = 0, scr_bytes = 0;
  bool demag_ready = false;
  // persistent offsets
  size_t off_table, off_wx, off_wy, off_wz, off_posz, off_fz, off_fx, off_fy, off_posx, off_posy, off_t2x, off_t2y, off_t2z, off_rkstate, off_bbstate, off_bbpart, pers_need;
  // scratch offsets
  size_t off_a1, off_a2, off_hd, off_msa, off_msb, off_acc, off_sin, off_sout, off_rkf, off_emb_m, off_emb_h, off_mscaled, scr_need;
  RkfState rk_host{};
  bool rk_ready = false;
  bool bb_ready = false;
  unsigned long long launches = 0;
  // mm_rk_steps: a captured chunk of RK4 steps, valid for (m, dt, chunk length, settings epoch)
  unsigned long long epoch = 0;          // bumped by every call that changes what a step computes
  cudaGraphExec_t rk_graph = nullptr;
  cudaStream_t rk_capture_stream = nullptr;
  void* rk_graph_m = nullptr;
  double rk_graph_dt = 0;
  int rk_graph_steps = 0;
  unsigned long long rk_graph_epoch = 0, rk_graph_launches = 0;
  // mm_llg_rhs_host_batch: copy streams and the events that order the two staging slots
  cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
  Prof prof;
  double prof_ms[Prof::kKinds] = {0};
  unsigned long long prof_cnt[Prof::kKinds] = {0};
  char err[256] = "";
};

static mm_status fail(mm_ctx* c, mm_status s, const char* fmt, ...) {
  char* dst = c ? c->err : g_create_error;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 256, fmt, ap);
  va_end(ap);
  return s;
}

static size_t align256(size_t v) { return (v + 255) / 256 * 256; }
static int padded(int n) { return n == 1 ? 1 : 2 * n; }

// Tile width: the largest divisor of `extent` (the tiled axis: tiles are never ragged) that is
// at most `cap` and fits the shared-memory budget.  Powers of two give a power of two.
static int pick_tile(int extent, size_t bytes_per_col, size_t budget, int cap) {
  int best = 1;
  for (int b = 2; b <= extent && b <= cap && (size_t)b * bytes_per_col <= budget; ++b)
    if (extent % b == 0) best = b;
  return best;
}
// n = 2^a 3^b 5^c 7^d (the radices of fft_core.cuh)
static bool smooth7(int n) { return n >= 1 && make_plan(n).nstages >= 0; }

// Tile widths and workspace layout; called at create and again if tiles change.
// Embedding: a mesh the power-of-two kernels do not cover is placed in the corner of
// the next mesh they do cover (cells outside carry no magnetisation and add nothing to eq. 4), when the
// extra cells cost less than the slower generic passes.  Per-cell cost ratio generic / fast measured on
// the paper's meshes (profiles/r01_v4_paper_meshes.md): about 4.6 in fp32, 3.1 in fp64.
static bool embed_mesh(const mm_ctx* c, int* ex, int* ey, int* ez) {
  // smallest length the x-first kernels cover that holds n (0: none)
  static const int kxy[] = {64, 100, 128, 256, 350, 400, 512, 1024};
  auto up = [](int n, const int* list, int count) { for (int i = 0; i < count; ++i) if (list[i] >= n) return list[i]; return 0; };
  const int x = up(c->nx, kxy, 8), y = up(c->ny, kxy, 8);
  int z = 0;
  const int zc[] = {c->nz, c->nz + 1, 16, 350, 400};
  for (int v : zc)
    if (!z && v >= c->nz && fast_z_transform(v, c->es, 4)) z = v;
  if (!x || !y || !z || !fast_supported(x, y, z, c->es)) return false;
  const double r = (double)x * y * z / ((double)c->nx * c->ny * c->nz);
  // fp64 with nz' = 256 runs the wide-pencil K3 at 0.34 of the roofline: a smaller margin
  if (r > (c->es == 4 ? 3.0 : (z == 256 ? 1.7 : 2.2))) return false;
  *ex = x; *ey = y; *ez = z;
  return true;
}

static void plan_layout(mm_ctx* c) {
  DemagGeom& g = c->geom;
  c->dnx = c->nx; c->dny = c->ny; c->dnz = c->nz;
  c->embed = c->path_pref == 0 && !fast_supported(c->nx, c->ny, c->nz, c->es) && embed_mesh(c, &c->dnx, &c->dny, &c->dnz);
  g.nx = c->dnx; g.ny = c->dny; g.nz = c->dnz;
  c->fast = c->path_pref != 1 && c->path_pref != 3 && fast_supported(c->dnx, c->dny, c->dnz, c->es);
  // x-first kernels: the z transform may be longer than 2 nz (any period >= 2 nz - 1 yields the same linear
  // convolution, reading Q27); the table and the z twiddles follow the transform
  c->nzt = c->fast ? fast_z_transform(c->dnz, c->es, c->dny) : c->dnz;
  g.Px = padded(c->dnx); g.Py = padded(c->dny); g.Pz = padded(c->nzt);
  g.Kz = g.Pz == 1 ? 1 : g.Pz / 2 + 1;
  g.px = make_plan(c->dnx); g.py = make_plan(c->dny); g.pz = make_plan(c->dnz);
  const size_t cs = 2 * c->es;
  const size_t kMax = 200 * 1024;  // usable dynamic shared memory we plan for (227 KB limit)
  g.Bz = c->want_bz ? c->want_bz : pick_tile(c->dnx, 3 * g.Pz * cs, 100 * 1024, 32);
  g.By = c->want_by ? c->want_by : pick_tile(c->dnx, g.Py * cs, 100 * 1024, 32);
  // two ky' rows per x-pass tile: small tiles, several CTAs per SM (measured best on 256x256x32, 350^3, 400^3)
  g.Bk = c->want_bk ? c->want_bk : pick_tile(g.Py, 3 * g.Px * cs, kMax, 2);
  if (g.Bz > c->dnx) g.Bz = c->dnx;
  if (g.By > c->dnx) g.By = c->dnx;
  if (g.Bk > g.Py) g.Bk = g.Py;
  InitGeom& ig = c->igeom;
  ig.nx = c->dnx; ig.ny = c->dny; ig.nz = c->dnz;
  ig.Px = g.Px; ig.Py = g.Py; ig.Pz = g.Pz; ig.Kz = g.Kz;
  ig.ox = c->dnx == 1 ? 1 : c->dnx + 1;
  ig.oy = c->dny == 1 ? 1 : c->dny + 1;
  ig.oz = c->nzt == 1 ? 1 : c->nzt + 1;
  ig.ozp = (ig.oz + 1) / 2 * 2;
  ig.Bk = g.Bk;
  // measured (profiles/r01_v4_paper_meshes.md): the mixed-radix x-first kernels only tie with the generic
  // z-first passes, so they are opt-in (path 3) until their stages move into registers
  c->mixed = c->path_pref == 3 && mixed_supported(c->dnx, c->dny, c->dnz, c->es);
  FastGeom& fg = c->fgeom;
  fg.nx = c->dnx; fg.ny = c->dny; fg.nz = c->dnz; fg.nzt = c->nzt;
  fg.Px = g.Px; fg.Py = g.Py; fg.Pz = g.Pz;
  fg.Q = 3 * c->dnz;
  // persistent
  size_t o = 0;
  c->off_table = o;
  o += c->xfirst() ? align256((size_t)ig.ox * ig.oy * ig.ozp * 6 * c->es)
               : align256((size_t)g.Kz * g.Py * g.Px * 6 * c->es);
  c->off_wx = o; o += align256((size_t)g.Px * cs);
  c->off_wy = o; o += align256((size_t)g.Py * cs);
  c->off_wz = o; o += align256((size_t)g.Pz * cs);
  c->off_posz = o; o += align256((size_t)g.Pz * 2);
  c->off_fz = o; o += align256((size_t)g.Pz * 2);
  c->off_fx = o; o += align256((size_t)g.Px * 2);
  c->off_fy = o; o += align256((size_t)g.Py * 2);
  c->off_posx = o; o += align256((size_t)g.Px * 2);
  c->off_posy = o; o += align256((size_t)g.Py * 2);
  c->off_t2x = o; o += align256((size_t)g.Px * cs);
  c->off_t2y = o; o += align256((size_t)g.Py * cs);
  c->off_t2z = o; o += align256((size_t)g.Pz * cs);
  c->off_rkstate = o; o += align256(sizeof(RkfState));
  c->off_bbstate = o; o += align256(sizeof(BbState));
  c->off_bbpart = o; o += align256((size_t)kBbMaxBlocks * 3 * sizeof(double));
  c->pers_need = o;
  // scratch
  const size_t n3 = (size_t)c->nx * c->ny * c->nz * 3 * c->es;
  o = 0;
  if (c->fast && c->slabs) {   // S_r[rpr][nx][Q] and A2_r[rpr][Px][Q] of every rank, back to back
    const size_t rows = (size_t)c->slabs * c->slab_rpr();
    c->off_a1 = o; o += align256(rows * g.nx * fg.Q * cs);
    c->off_a2 = o; o += align256(rows * g.Px * fg.Q * cs);
  } else if (c->xfirst()) {
    const size_t planes2 = c->dnx + 1;
    c->off_a1 = o; o += align256((size_t)(c->dnx + 1) * g.ny * fg.Q * cs);
    c->off_a2 = o; o += align256(planes2 * g.Py * fg.Q * cs);
  } else {
    c->off_a1 = o; o += align256((size_t)3 * g.Kz * g.ny * g.nx * cs);
    c->off_a2 = o; o += align256((size_t)3 * g.Kz * g.Py * g.nx * cs);
  }
  const size_t spectra = o;
  c->off_hd = o; o += align256(n3);
  c->off_msa = o; o += align256(n3);
  c->off_msb = o; o += align256(n3);
  c->off_acc = o; o += align256(n3);
  c->off_sin = o; o += align256(n3);
  c->off_sout = o; o += align256(n3);
  c->off_rkf = o; o += 6 * align256(n3);
  const size_t e3 = c->embed ? (size_t)c->dnx * c->dny * c->dnz * 3 * c->es : 0;   // embedded m and H
  c->off_emb_m = o; o += align256(e3);
  c->off_emb_h = o; o += align256(e3);
  c->off_mscaled = o; o += align256(n3);   // M = Ms_i m when Ms varies per cell   // RKF45: k_1..k_6, n3 reals apart (stage state and candidate reuse msa, msb)
  (void)spectra;
  const size_t init_need = demag_init_scratch_bytes(ig);  // aliases the start of scratch
  c->scr_need = o > init_need ? o : init_need;
}

extern "C" {

mm_status mm_ctx_create(int nx, int ny, int nz, double dx, double dy, double dz, mm_dtype dtype,
                        mm_ctx** out) {
  if (!out) return fail(nullptr, MM_ERR_INVALID_ARG, "mm_ctx_create: out is NULL");
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0))
    return fail(nullptr, MM_ERR_INVALID_ARG, "mm_ctx_create: sizes and cell lengths must be positive");
  if (dtype != MM_F32 && dtype != MM_F64)
    return fail(nullptr, MM_ERR_INVALID_ARG, "mm_ctx_create: unknown dtype %d", (int)dtype);
  if (nx > 1024 || ny > 1024 || nz > 512 || !smooth7(nx) || !smooth7(ny) || !smooth7(nz))
    return fail(nullptr, MM_ERR_UNSUPPORTED_SIZE,
                "mm_ctx_create: %dx%dx%d unsupported (each n must be of the form 2^a 3^b 5^c 7^d, "
                "nx,ny <= 1024, nz <= 512)", nx, ny, nz);
  mm_ctx* c = new (std::nothrow) mm_ctx();
  if (!c) return fail(nullptr, MM_ERR_INVALID_ARG, "mm_ctx_create: out of host memory");
  c->nx = nx; c->ny = ny; c->nz = nz;
  c->dx = dx; c->dy = dy; c->dz = dz;
  c->dtype = dtype;
  c->es = dtype == MM_F32 ? 4 : 8;
  plan_layout(c);
  *out = c;
  return MM_OK;
}

mm_status mm_ctx_destroy(mm_ctx* ctx) {
  if (ctx) {
    if (ctx->rk_graph) cudaGraphExecDestroy(ctx->rk_graph);
    if (ctx->rk_capture_stream) cudaStreamDestroy(ctx->rk_capture_stream);
    if (ctx->h2d_stream) cudaStreamDestroy(ctx->h2d_stream);
    if (ctx->d2h_stream) cudaStreamDestroy(ctx->d2h_stream);
    for (int i = 0; i < 2; ++i) {
      if (ctx->ev_in[i]) cudaEventDestroy(ctx->ev_in[i]);
      if (ctx->ev_comp[i]) cudaEventDestroy(ctx->ev_comp[i]);
      if (ctx->ev_out[i]) cudaEventDestroy(ctx->ev_out[i]);
    }
  }
  delete ctx;
  return MM_OK;
}

mm_status mm_ctx_set_stream(mm_ctx* ctx, void* cuda_stream) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  ctx->stream = static_cast<cudaStream_t>(cuda_stream);
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_ctx_set_tiles(mm_ctx* ctx, int bz, int by, int bk) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (ctx->pers) return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_tiles: call before mm_ctx_set_workspace");
  const int v[3] = {bz, by, bk};
  for (int i = 0; i < 3; ++i)
    if (v[i] < 0 || v[i] > 64)
      return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_tiles: tile widths must be in 0 .. 64");
  if ((bz && ctx->nx % bz) || (by && ctx->nx % by) || (bk && padded(ctx->ny) % bk))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_tiles: bz, by must divide nx and bk must divide the padded ny");
  ctx->want_bz = bz; ctx->want_by = by; ctx->want_bk = bk;
  plan_layout(ctx);
  const size_t cs = 2 * ctx->es;
  const DemagGeom& g = ctx->geom;
  const size_t lim = 227 * 1024;
  if ((size_t)3 * g.Pz * g.Bz * cs > lim || (size_t)g.Py * g.By * cs > lim ||
      (size_t)3 * g.Px * g.Bk * cs > lim) {
    ctx->want_bz = ctx->want_by = ctx->want_bk = 0;
    plan_layout(ctx);
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_tiles: tile exceeds 227 KB of shared memory");
  }
  return MM_OK;
}

mm_status mm_ctx_set_path(mm_ctx* ctx, int path) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (ctx->pers) return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_path: call before mm_ctx_set_workspace");
  if (path < 0 || path > 3)
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_path: path must be 0 .. 3");
  if (path == 3 && !mixed_supported(ctx->nx, ctx->ny, ctx->nz, ctx->es))
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_ctx_set_path: the mixed-radix x-first kernels do not cover %dx%dx%d",
                ctx->nx, ctx->ny, ctx->nz);
  if (path == 2 && !fast_supported(ctx->nx, ctx->ny, ctx->nz, ctx->es))
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_ctx_set_path: the fast kernels do not cover %dx%dx%d",
                ctx->nx, ctx->ny, ctx->nz);
  ctx->path_pref = path;
  plan_layout(ctx);
  return MM_OK;
}

mm_status mm_ctx_path(const mm_ctx* ctx, int* path) {
  if (!ctx || !path) return MM_ERR_INVALID_ARG;
  *path = ctx->fast ? (ctx->embed ? 3 : 1) : (ctx->mixed ? 2 : 0);
  return MM_OK;
}

mm_status mm_ctx_set_slabs(mm_ctx* ctx, int ranks) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (ctx->pers) return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_slabs: call before mm_ctx_set_workspace");
  if (ranks < 0 || ranks > 8) return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_slabs: ranks must be 0 .. 8");
  if (ranks && !(ctx->fast && !ctx->embed && fast_two_stage(ctx->nx) && fast_two_stage(ctx->ny) && ranks <= ctx->nx))
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_ctx_set_slabs: the slab layout needs a mesh the x-first kernels cover "
                "with two-stage plans along x and y (%dx%dx%d does not qualify)", ctx->nx, ctx->ny, ctx->nz);
  ctx->slabs = ranks;
  plan_layout(ctx);
  return MM_OK;
}

mm_status mm_ctx_workspace_bytes(const mm_ctx* ctx, size_t* persistent, size_t* scratch) {
  if (!ctx || !persistent || !scratch) return MM_ERR_INVALID_ARG;
  *persistent = ctx->pers_need;
  *scratch = ctx->scr_need;
  return MM_OK;
}

mm_status mm_ctx_set_workspace(mm_ctx* ctx, void* persistent, size_t pbytes, void* scratch,
                               size_t sbytes) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!persistent || !scratch || ((uintptr_t)persistent & 255) || ((uintptr_t)scratch & 255))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_ctx_set_workspace: NULL or not 256-byte aligned");
  if (pbytes < ctx->pers_need || sbytes < ctx->scr_need)
    return fail(ctx, MM_ERR_WORKSPACE, "mm_ctx_set_workspace: need %zu + %zu bytes, got %zu + %zu",
                ctx->pers_need, ctx->scr_need, pbytes, sbytes);
  ctx->pers = static_cast<unsigned char*>(persistent);
  ctx->scr = static_cast<unsigned char*>(scratch);
  ctx->pers_bytes = pbytes;
  ctx->scr_bytes = sbytes;
  ctx->demag_ready = false;
  ctx->rk_ready = false;
  ctx->bb_ready = false;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_material(mm_ctx* ctx, double Ms, double Aex, double Ku, const double axis[3],
                          double alpha, double gamma) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!(Ms > 0) || Aex < 0 || alpha < 0 || !(gamma > 0))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_material: need Ms > 0, Aex >= 0, alpha >= 0, gamma > 0");
  double u[3] = {0, 0, 1};
  if (Ku != 0.0) {
    if (!axis) return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_material: Ku != 0 needs an axis");
    const double n = std::sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (!(n > 0)) return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_material: zero anisotropy axis");
    for (int i = 0; i < 3; ++i) u[i] = axis[i] / n;
  }
  ctx->Ms = Ms; ctx->Aex = Aex; ctx->Ku = Ku;
  for (int i = 0; i < 3; ++i) ctx->axis[i] = u[i];
  ctx->alpha = alpha; ctx->gamma = gamma;
  ctx->have_material = true;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_zeeman(mm_ctx* ctx, const double Hext[3]) {
  if (!ctx || !Hext) return MM_ERR_INVALID_ARG;
  for (int i = 0; i < 3; ++i) ctx->Hext[i] = Hext[i];
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_dmi(mm_ctx* ctx, double D, const double e[9]) {
  if (!ctx || !e) return MM_ERR_INVALID_ARG;
  for (int i = 0; i < 9; ++i)
    if (!std::isfinite(e[i])) return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_dmi: DMI vectors must be finite");
  if (!std::isfinite(D)) return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_dmi: D must be finite");
  ctx->Ddmi = D;
  for (int i = 0; i < 9; ++i) ctx->edmi[i] = e[i];
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_stt(mm_ctx* ctx, const double p[3], double a_damp, double a_field) {
  if (!ctx || !p) return MM_ERR_INVALID_ARG;
  const double n = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
  if (!(n > 0) || !std::isfinite(n) || !std::isfinite(a_damp) || !std::isfinite(a_field))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_stt: need a non-zero polarisation and finite amplitudes");
  for (int i = 0; i < 3; ++i) ctx->stt_p[i] = p[i] / n;
  ctx->stt_damp = a_damp;
  ctx->stt_field = a_field;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_material_cells(mm_ctx* ctx, const void* Ms_cells, const void* A_cells) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (((uintptr_t)Ms_cells & 15) || ((uintptr_t)A_cells & 15))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_material_cells: device pointers must be 16-byte aligned");
  ctx->ms_cells = Ms_cells;
  ctx->a_cells = A_cells;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_set_terms(mm_ctx* ctx, unsigned term_mask) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (term_mask & ~63u) return fail(ctx, MM_ERR_INVALID_ARG, "mm_set_terms: unknown term bits 0x%x", term_mask);
  ctx->terms = term_mask;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_ctx_launch_count(const mm_ctx* ctx, unsigned long long* count) {
  if (!ctx || !count) return MM_ERR_INVALID_ARG;
  *count = ctx->launches;
  return MM_OK;
}

const char* mm_last_error(const mm_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

const char* mm_ctx_kernel_name(const mm_ctx* ctx, int kind) {
  if (!ctx || kind < 0 || kind > 5) return "";
  if (kind == 5) {
    if (ctx->ms_cells || ctx->a_cells) return "pw_inhom_kernel";
    return ctx->nz % 2 == 0 ? "pw_vec_kernel" : "pw_cell_kernel";
  }
  if (ctx->fast) {
    const bool two_x = fast_two_stage(ctx->dnx), two_y = fast_two_stage(ctx->dny);
    switch (kind) {
      case 0: return two_x ? (strided_tma_x_usable(ctx->dnx, ctx->dny, 3 * ctx->dnz, ctx->es) ? "xf2_tma_kernel" : "xf2_kernel")
                           : (strided_tma3_x_usable(ctx->dny, 3 * ctx->dnz, ctx->es) ? "xf3_tma_kernel" : "xf_fast_kernel");
      case 1: return two_y ? (strided_tma_usable(ctx->dny, 3 * ctx->dnz, ctx->es, 1) ? "yf2_tma_kernel" : "yf2_kernel")
                           : (strided_tma_usable(ctx->dny, 3 * ctx->dnz, ctx->es, 1) ? "yf3_tma_kernel" : "yf_fast_kernel");
      case 2: return ctx->nzt == 256 ? "zw_fast_kernel" : (ctx->nzt > 256 ? "zt_kernel" : "zp_fast_kernel");
      case 3: return two_y ? (strided_tma_usable(ctx->dny, 3 * ctx->dnz, ctx->es, 3) ? "yi2_tma_kernel" : "yi2_kernel")
                           : (strided_tma_usable(ctx->dny, 3 * ctx->dnz, ctx->es, 3) ? "yi3_tma_kernel" : "yi_fast_kernel");
      default: return two_x ? (strided_tma_x_usable(ctx->dnx, ctx->dny, 3 * ctx->dnz, ctx->es) ? "xi2_tma_kernel" : "xi2_kernel")
                            : (strided_tma3_x_usable(ctx->dny, 3 * ctx->dnz, ctx->es) ? "xi3_tma_kernel" : "xi_fast_kernel");
    }
  }
  static const char* const mixed[5] = {"xf_mixed_kernel", "yf_mixed_kernel", "zp_mixed_kernel", "yi_mixed_kernel",
                                       "xi_mixed_kernel"};
  static const char* const generic[5] = {"zf_kernel", "yf_kernel", "xp_kernel", "yi_kernel", "zi_kernel"};
  return ctx->mixed ? mixed[kind] : generic[kind];
}

mm_status mm_ctx_set_profiling(mm_ctx* ctx, int enable) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  ctx->prof.on = enable != 0;
  ++ctx->epoch;
  return MM_OK;
}

mm_status mm_ctx_kernel_times(mm_ctx* ctx, int reset, double ms_sum[8], unsigned long long count[8]) {
  if (!ctx || !ms_sum || !count) return MM_ERR_INVALID_ARG;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) { snprintf(ctx->err, 256, "mm_ctx_kernel_times: %s", cudaGetErrorString(e)); return MM_ERR_CUDA; }
  Prof& p = ctx->prof;
  for (int i = 0; i + 1 < p.n; ++i) {
    if (p.kind[i] < 0) continue;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, p.ev[i], p.ev[i + 1]) == cudaSuccess) {
      ctx->prof_ms[p.kind[i]] += ms;
      ctx->prof_cnt[p.kind[i]] += 1;
    }
  }
  p.n = 0;
  for (int k = 0; k < Prof::kKinds; ++k) {
    ms_sum[k] = ctx->prof_ms[k];
    count[k] = ctx->prof_cnt[k];
    if (reset) { ctx->prof_ms[k] = 0; ctx->prof_cnt[k] = 0; }
  }
  return MM_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ internals

static mm_status cuda_fail(mm_ctx* c, const char* what, cudaError_t e) {
  return fail(c, MM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

template <typename T> static void fill_twiddles(std::vector<unsigned char>& buf, size_t off, int P) {
  Cx<T>* w = reinterpret_cast<Cx<T>*>(buf.data() + off);
  for (int q = 0; q < P; ++q) {
    // exact octant reduction through the integer phase keeps the table symmetric
    const long double ph = -2.0L * 3.14159265358979323846264338327950288L * (long double)q / (long double)P;
    w[q] = mk<T>((T)cosl(ph), (T)sinl(ph));
  }
}

// Wt[bf K1 + k1] = exp(-2 pi i bf k1 / P) of the two-stage plan of length L = P / 2 (demag_fast2.cu).
template <typename T> static void fill_twiddles2(std::vector<unsigned char>& buf, size_t off, int L) {
  int K1, K2;
  fast2_plan(L, &K1, &K2);
  const int P = 2 * L;
  Cx<T>* w = reinterpret_cast<Cx<T>*>(buf.data() + off);
  for (int bf = 0; bf < K2; ++bf)
    for (int k1 = 0; k1 < K1; ++k1) {
      const int q = (bf * k1) % P;
      const long double ph = -2.0L * 3.14159265358979323846264338327950288L * (long double)q / (long double)P;
      w[bf * K1 + k1] = mk<T>((T)cosl(ph), (T)sinl(ph));
    }
}

template <typename T> static mm_status demag_init_t(mm_ctx* c) {
  const DemagGeom& g = c->geom;
  // small tables: twiddles and digit-reversal maps, built on the host, uploaded once.  The upload stops
  // short of the RKF45 / minimiser controller records, which mm_rkf45_init / mm_minimize_init own and
  // may have written already (the header does not fix the order of the init calls).
  const size_t small_off = c->off_wx, small_bytes = c->off_rkstate - c->off_wx;
  std::vector<unsigned char> host(small_bytes, 0);
  fill_twiddles<T>(host, c->off_wx - small_off, g.Px);
  fill_twiddles<T>(host, c->off_wy - small_off, g.Py);
  fill_twiddles<T>(host, c->off_wz - small_off, g.Pz);
  const bool two_x = c->fast && fast_two_stage(c->dnx), two_y = c->fast && fast_two_stage(c->dny);
  if (two_x) fill_twiddles2<T>(host, c->off_t2x - small_off, c->dnx);
  if (two_y) fill_twiddles2<T>(host, c->off_t2y - small_off, c->dny);
  if (c->fast && ztile_supported(c->nzt)) fill_twiddles2<T>(host, c->off_t2z - small_off, c->nzt);
  auto u16 = [&](size_t off) { return reinterpret_cast<uint16_t*>(host.data() + (off - small_off)); };
  for (int k = 0; k < g.Pz; ++k) {
    const int p = pos_of_freq(g.pz, k);
    u16(c->off_posz)[k] = (uint16_t)p;
    u16(c->off_fz)[p] = (uint16_t)k;
  }
  for (int k = 0; k < g.Px; ++k) {
    const int p = pos_of_freq(g.px, k);
    u16(c->off_posx)[k] = (uint16_t)(c->fast ? (two_x ? k : fast_swizzle(c->dnx, fast_pos_logical(c->dnx, k))) : p);
    u16(c->off_fx)[p] = (uint16_t)k;
  }
  for (int k = 0; k < g.Py; ++k) {
    const int p = pos_of_freq(g.py, k);
    u16(c->off_posy)[k] = (uint16_t)(c->fast ? (two_y ? k : fast_pos_logical(c->dny, k)) : p);
    u16(c->off_fy)[p] = (uint16_t)k;
  }
  cudaError_t e = cudaMemcpyAsync(c->pers + small_off, host.data(), small_bytes,
                                  cudaMemcpyHostToDevice, c->stream);
  if (e != cudaSuccess) return cuda_fail(c, "mm_demag_init: table upload", e);
  e = demag_init_launch<T>(c->igeom, c->dx, c->dy, c->dz, c->scr,
                           reinterpret_cast<const uint16_t*>(c->pers + c->off_fx),
                           reinterpret_cast<const uint16_t*>(c->pers + c->off_fy),
                           reinterpret_cast<T*>(c->pers + c->off_table), c->xfirst() ? ((c->fast && c->slabs) ? 2 : 1) : 0,
                           c->stream, &c->launches);
  if (e != cudaSuccess) return cuda_fail(c, "mm_demag_init: launch", e);
  e = cudaStreamSynchronize(c->stream);  // also keeps `host` alive until the copy is done
  if (e != cudaSuccess) return cuda_fail(c, "mm_demag_init: execution", e);
  c->demag_ready = true;
  return MM_OK;
}

template <typename T> static DemagBufs<T> bufs_of(mm_ctx* c) {
  DemagBufs<T> b;
  b.Wx = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wx);
  b.Wy = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wy);
  b.Wz = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wz);
  b.posz = reinterpret_cast<const uint16_t*>(c->pers + c->off_posz);
  b.table = reinterpret_cast<const T*>(c->pers + c->off_table);
  b.A1 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a1);
  b.A2 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a2);
  return b;
}

template <typename T> static PwParams<T> pw_of(const mm_ctx* c, unsigned terms) {
  PwParams<T> p{};
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
  p.terms = terms;
  const double pe = 2.0 * c->Aex / (kMu0 * c->Ms);
  p.ex[0] = (T)(pe / (c->dx * c->dx));
  p.ex[1] = (T)(pe / (c->dy * c->dy));
  p.ex[2] = (T)(pe / (c->dz * c->dz));
  p.kan = (T)(2.0 * c->Ku / (kMu0 * c->Ms));
  for (int i = 0; i < 3; ++i) { p.u[i] = (T)c->axis[i]; p.hext[i] = (T)c->Hext[i]; }
  const double pd = 2.0 * c->Ddmi / (kMu0 * c->Ms);
  const double cell[3] = {c->dx, c->dy, c->dz};
  const int nn[3] = {c->nx, c->ny, c->nz};
  for (int k = 0; k < 3; ++k)
    for (int i = 0; i < 3; ++i) p.dmi[k][i] = nn[k] > 1 ? (T)(pd * c->edmi[3 * k + i] / (2.0 * cell[k])) : (T)0;
  p.ms_cells = static_cast<const T*>(c->ms_cells);
  p.a_cells = static_cast<const T*>(c->a_cells);
  p.ms_ref = (T)c->Ms; p.a_ref = (T)c->Aex;
  for (int k = 0; k < 3; ++k) {
    p.exq[k] = (T)(2.0 / (kMu0 * cell[k] * cell[k]));
    for (int i = 0; i < 3; ++i)
      p.dmiq[k][i] = nn[k] > 1 ? (T)(2.0 * c->Ddmi / kMu0 * c->edmi[3 * k + i] / (2.0 * cell[k])) : (T)0;
  }
  p.kanq = (T)(2.0 * c->Ku / kMu0);
  for (int i = 0; i < 3; ++i) p.sp[i] = (T)c->stt_p[i];
  p.sdamp = (T)c->stt_damp; p.sfield = (T)c->stt_field;
  p.pref = (T)(-c->gamma / (1.0 + c->alpha * c->alpha));
  p.alpha = (T)c->alpha;
  p.first = 0; p.wk = (T)1; p.a = (T)0;
  return p;
}

static mm_status check_ptr(mm_ctx* c, const char* fn, const void* a, const void* b) {
  if (!a || !b || ((uintptr_t)a & 15) || ((uintptr_t)b & 15))
    return fail(c, MM_ERR_INVALID_ARG, "%s: NULL or not 16-byte aligned device pointer", fn);
  return MM_OK;
}

static mm_status need_ready(mm_ctx* c, const char* fn, bool demag) {
  if (!c->have_material) return fail(c, MM_ERR_NOT_INITIALISED, "%s: mm_set_material not called", fn);
  if (!c->scr || !c->pers) return fail(c, MM_ERR_NOT_INITIALISED, "%s: mm_ctx_set_workspace not called", fn);
  if (demag && !c->demag_ready) return fail(c, MM_ERR_NOT_INITIALISED, "%s: mm_demag_init not called", fn);
  return MM_OK;
}

template <typename T> static FastBufs<T> fast_bufs_of(mm_ctx* c) {
  FastBufs<T> b;
  b.Wx = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wx);
  b.Wy = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wy);
  b.Wz = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wz);
  b.posx = reinterpret_cast<const uint16_t*>(c->pers + c->off_posx);
  b.posy = reinterpret_cast<const uint16_t*>(c->pers + c->off_posy);
  b.T2x = reinterpret_cast<const Cx<T>*>(c->pers + c->off_t2x);
  b.T2y = reinterpret_cast<const Cx<T>*>(c->pers + c->off_t2y);
  b.T2z = reinterpret_cast<const Cx<T>*>(c->pers + c->off_t2z);
  b.two_x = fast_two_stage(c->dnx);
  b.two_y = fast_two_stage(c->dny);
  b.table = reinterpret_cast<const T*>(c->pers + c->off_table);
  b.A1 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a1);
  b.A2 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a2);
  return b;
}

template <typename T> static MixedBufs<T> mixed_bufs_of(mm_ctx* c) {
  MixedBufs<T> b;
  b.Wx = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wx);
  b.Wy = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wy);
  b.Wz = reinterpret_cast<const Cx<T>*>(c->pers + c->off_wz);
  b.posx = reinterpret_cast<const uint16_t*>(c->pers + c->off_posx);
  b.posy = reinterpret_cast<const uint16_t*>(c->pers + c->off_posy);
  b.fz = reinterpret_cast<const uint16_t*>(c->pers + c->off_fz);
  b.table = reinterpret_cast<const T*>(c->pers + c->off_table);
  b.A1 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a1);
  b.A2 = reinterpret_cast<Cx<T>*>(c->scr + c->off_a2);
  return b;
}

template <typename T> static mm_status demag_t(mm_ctx* c, const void* m, void* H);

// Slab decomposition emulated on one device (mm_ctx_set_slabs): per rank the y pass of its x
// planes (stores go to the owners of the spectrum rows: the first transpose), then per rank x forward, z . Nhat .
// z^-1 and x inverse on its own ky rows, then per rank the inverse y pass of its x planes (loads come from the
// owners: the second transpose).  On R GPUs every "for r" body is what rank r enqueues, with peer pointers in sv.p.
template <typename T> static mm_status demag_slab_t(mm_ctx* c, const T* m, T* H) {
  const FastGeom& g = c->fgeom;
  const FastBufs<T> b = fast_bufs_of<T>(c);
  const int R = c->slabs, rpr = c->slab_rpr(), rows_all = g.ny + 1;
  const size_t s_stride = (size_t)rpr * g.nx * g.Q, a2_stride = (size_t)rpr * g.Px * g.Q;
  SlabView<T> sv{};
  for (int r = 0; r < R; ++r) sv.p[r] = b.A1 + r * s_stride;
  sv.rpr = rpr; sv.nx = g.nx;
  cudaError_t e = cudaSuccess;
  auto x_first = [&](int r) { return (int)((long long)r * g.nx / R); };
  for (int r = 0; r < R && e == cudaSuccess; ++r) {
    sv.x0 = x_first(r);
    c->prof.mark(0, c->stream);
    e = slab_y_launch<T>(0, g.ny, x_first(r + 1) - sv.x0, g.Q, b.T2y, sv, m, H, (T)(-c->Ms), c->stream);
    ++c->launches;
  }
  for (int r = 0; r < R && e == cudaSuccess; ++r) {
    const int rows = rows_all - r * rpr < rpr ? rows_all - r * rpr : rpr;   // ky rows this rank owns
    if (rows <= 0) break;
    FastGeom gx = g;            // the x transform of rank r: `rows` planes of [nx][Q], transform length nx
    gx.nx = rows - 1; gx.ny = g.nx; gx.Py = g.Px;
    FastBufs<T> bx = b;
    bx.A1 = b.A1 + r * s_stride; bx.A2 = b.A2 + r * a2_stride; bx.T2y = b.T2x; bx.posy = b.posx;
    c->prof.mark(1, c->stream);
    e = strided_tma_launch<T>(1, gx, bx, c->stream);
    if (e == cudaErrorNotSupported) e = strided2_launch<T>(1, gx, bx, m, H, (T)0, c->stream);
    if (e != cudaSuccess) break;
    c->prof.mark(2, c->stream);
    if ((e = k3_launch<T>(gx, bx, r * rpr, rows, 1, c->stream)) != cudaSuccess) break;
    c->prof.mark(3, c->stream);
    e = strided_tma_launch<T>(3, gx, bx, c->stream);
    if (e == cudaErrorNotSupported) e = strided2_launch<T>(3, gx, bx, m, H, (T)0, c->stream);
    c->launches += 3;
  }
  for (int r = 0; r < R && e == cudaSuccess; ++r) {
    sv.x0 = x_first(r);
    c->prof.mark(4, c->stream);
    e = slab_y_launch<T>(4, g.ny, x_first(r + 1) - sv.x0, g.Q, b.T2y, sv, m, H, (T)(-c->Ms), c->stream);
    ++c->launches;
  }
  c->prof.mark(-1, c->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "demag (slab layout) launch", e);
}

// per-cell Ms: the passes transform M = Ms_i m and the final scale is -1 (eq. 4 with M = Ms m)
template <typename T> static mm_status demag_cells_t(mm_ctx* c, const void* m, void* H) {
  T* M = reinterpret_cast<T*>(c->scr + c->off_mscaled);
  cudaError_t e = scale_by_ms_launch<T>(static_cast<const T*>(m), static_cast<const T*>(c->ms_cells), M,
                                        (size_t)c->nx * c->ny * c->nz, c->stream);
  if (e != cudaSuccess) return cuda_fail(c, "demag (per-cell Ms) launch", e);
  ++c->launches;
  const double Ms = c->Ms;
  const void* cells = c->ms_cells;
  c->Ms = 1.0; c->ms_cells = nullptr;
  const mm_status s = demag_t<T>(c, M, H);
  c->Ms = Ms; c->ms_cells = cells;
  return s;
}

template <typename T> static mm_status demag_t(mm_ctx* c, const void* m, void* H) {
  if (c->ms_cells) return demag_cells_t<T>(c, m, H);
  if (c->mixed) {
    const MixedPlans pl{c->geom.px, c->geom.py, c->geom.pz};
    cudaError_t e = demag_mixed_launch<T>(c->fgeom, pl, mixed_bufs_of<T>(c), static_cast<const T*>(m),
                                          static_cast<T*>(H), (T)(-c->Ms), c->stream, &c->launches, &c->prof);
    return e == cudaSuccess ? MM_OK : cuda_fail(c, "demag (mixed-radix path) launch", e);
  }
  if (c->fast && c->embed) {
    T* mE = reinterpret_cast<T*>(c->scr + c->off_emb_m);
    T* HE = reinterpret_cast<T*>(c->scr + c->off_emb_h);
    c->prof.mark(0, c->stream);
    cudaError_t e = embed_copy_launch<T>(static_cast<const T*>(m), mE, c->nx, c->ny, c->nz, c->dnx, c->dny, c->dnz, 1, c->stream);
    if (e == cudaSuccess)
      e = demag_fast_launch<T>(c->fgeom, fast_bufs_of<T>(c), mE, HE, (T)(-c->Ms), c->stream, &c->launches, &c->prof);
    c->prof.mark(4, c->stream);
    if (e == cudaSuccess)
      e = embed_copy_launch<T>(HE, static_cast<T*>(H), c->nx, c->ny, c->nz, c->dnx, c->dny, c->dnz, 0, c->stream);
    c->prof.mark(-1, c->stream);
    c->launches += 2;
    return e == cudaSuccess ? MM_OK : cuda_fail(c, "demag (embedded fast path) launch", e);
  }
  if (c->fast && c->slabs) return demag_slab_t<T>(c, static_cast<const T*>(m), static_cast<T*>(H));
  if (c->fast) {
    cudaError_t e = demag_fast_launch<T>(c->fgeom, fast_bufs_of<T>(c), static_cast<const T*>(m),
                                         static_cast<T*>(H), (T)(-c->Ms), c->stream, &c->launches,
                                         &c->prof);
    return e == cudaSuccess ? MM_OK : cuda_fail(c, "demag (fast path) launch", e);
  }
  cudaError_t e = demag_field_launch<T>(c->geom, bufs_of<T>(c), static_cast<const T*>(m),
                                        static_cast<T*>(H), (T)(-c->Ms), c->stream, &c->launches,
                                        &c->prof);
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "demag launch", e);
}

// H_eff-type evaluations: optional demag into scratch, then the fused pointwise pass.
template <typename T>
static mm_status eval_t(mm_ctx* c, int mode, const void* m, void* out, void* m0, const PwParams<T>& p) {
  T* Hd = reinterpret_cast<T*>(c->scr + c->off_hd);
  if (mode != PW_EXCHANGE && (p.terms & MM_TERM_DEMAG)) {
    mm_status s = demag_t<T>(c, m, Hd);
    if (s != MM_OK) return s;
  }
  cudaError_t e = pointwise_launch<T>(mode, p, static_cast<const T*>(m), Hd, static_cast<T*>(out),
                                      static_cast<T*>(m0), reinterpret_cast<T*>(c->scr + c->off_acc),
                                      c->stream, &c->launches, &c->prof);
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "pointwise launch", e);
}

template <typename T> static mm_status rk_t(mm_ctx* c, void* m, double dt) {
  T* msa = reinterpret_cast<T*>(c->scr + c->off_msa);
  T* msb = reinterpret_cast<T*>(c->scr + c->off_msb);
  PwParams<T> p = pw_of<T>(c, c->terms);
  mm_status s;
  p.first = 1; p.wk = (T)1; p.a = (T)(0.5 * dt);
  if ((s = eval_t<T>(c, PW_RK_STAGE, m, msa, m, p)) != MM_OK) return s;
  p.first = 0; p.wk = (T)2; p.a = (T)(0.5 * dt);
  if ((s = eval_t<T>(c, PW_RK_STAGE, msa, msb, m, p)) != MM_OK) return s;
  p.wk = (T)2; p.a = (T)dt;
  if ((s = eval_t<T>(c, PW_RK_STAGE, msb, msa, m, p)) != MM_OK) return s;
  p.a = (T)(dt / 6.0);
  return eval_t<T>(c, PW_RK_FINAL, msa, nullptr, m, p);
}

static mm_status dispatch_eval(mm_ctx* c, int mode, unsigned terms, const void* m, void* out) {
  if (c->dtype == MM_F32) return eval_t<float>(c, mode, m, out, nullptr, pw_of<float>(c, terms));
  return eval_t<double>(c, mode, m, out, nullptr, pw_of<double>(c, terms));
}

extern "C" {

mm_status mm_demag_init(mm_ctx* ctx) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->scr || !ctx->pers)
    return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_demag_init: mm_ctx_set_workspace not called");
  if (ctx->demag_ready) return MM_OK;
  return ctx->dtype == MM_F32 ? demag_init_t<float>(ctx) : demag_init_t<double>(ctx);
}

mm_status mm_demag_nhat_export(mm_ctx* ctx, void* out) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->demag_ready) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_demag_nhat_export: mm_demag_init not called");
  if (!out || ((uintptr_t)out & 15)) return fail(ctx, MM_ERR_INVALID_ARG, "mm_demag_nhat_export: bad pointer");
  if (ctx->fast && ctx->slabs)
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_demag_nhat_export: not available in the slab layout");
  if (ctx->fast && ctx->nzt != ctx->dnz)
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_demag_nhat_export: this context transforms z with period %d, not 2 nz; "
                "select the generic passes (mm_ctx_set_path 1) to export the table at period 2 n", 2 * ctx->nzt);
  if (ctx->embed)
    return fail(ctx, MM_ERR_UNSUPPORTED_SIZE, "mm_demag_nhat_export: this context holds the table of the enclosing "
                "%dx%dx%d mesh; select the generic passes (mm_ctx_set_path 1) to export the mesh's own table",
                ctx->dnx, ctx->dny, ctx->dnz);
  const uint16_t* posx = reinterpret_cast<const uint16_t*>(ctx->pers + ctx->off_posx);
  const uint16_t* posy = reinterpret_cast<const uint16_t*>(ctx->pers + ctx->off_posy);
  cudaError_t e;
  if (ctx->dtype == MM_F32)
    e = demag_export_launch<float>(ctx->igeom, reinterpret_cast<const float*>(ctx->pers + ctx->off_table),
                                   posx, posy, static_cast<float*>(out), ctx->xfirst() ? 1 : 0, ctx->stream,
                                   &ctx->launches);
  else
    e = demag_export_launch<double>(ctx->igeom, reinterpret_cast<const double*>(ctx->pers + ctx->off_table),
                                    posx, posy, static_cast<double*>(out), ctx->xfirst() ? 1 : 0, ctx->stream,
                                    &ctx->launches);
  return e == cudaSuccess ? MM_OK : cuda_fail(ctx, "mm_demag_nhat_export", e);
}

mm_status mm_demag_field(mm_ctx* ctx, const void* m, void* H) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_demag_field", m, H)) != MM_OK) return s;
  if (m == H) return fail(ctx, MM_ERR_INVALID_ARG, "mm_demag_field: H must not alias m");
  if ((s = need_ready(ctx, "mm_demag_field", true)) != MM_OK) return s;
  return ctx->dtype == MM_F32 ? demag_t<float>(ctx, m, H) : demag_t<double>(ctx, m, H);
}

mm_status mm_exchange_field(mm_ctx* ctx, const void* m, void* H) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_exchange_field", m, H)) != MM_OK) return s;
  if (m == H) return fail(ctx, MM_ERR_INVALID_ARG, "mm_exchange_field: H must not alias m");
  if (!ctx->have_material) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_exchange_field: mm_set_material not called");
  return dispatch_eval(ctx, PW_EXCHANGE, MM_TERM_EXCHANGE, m, H);
}

mm_status mm_dmi_field(mm_ctx* ctx, const void* m, void* H) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_dmi_field", m, H)) != MM_OK) return s;
  if (m == H) return fail(ctx, MM_ERR_INVALID_ARG, "mm_dmi_field: H must not alias m");
  if (!ctx->have_material) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_dmi_field: mm_set_material not called");
  return dispatch_eval(ctx, PW_HEFF, MM_TERM_DMI, m, H);
}

mm_status mm_heff(mm_ctx* ctx, const void* m, void* H) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_heff", m, H)) != MM_OK) return s;
  if (m == H) return fail(ctx, MM_ERR_INVALID_ARG, "mm_heff: H must not alias m");
  if ((s = need_ready(ctx, "mm_heff", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  return dispatch_eval(ctx, PW_HEFF, ctx->terms, m, H);
}

mm_status mm_llg_rhs(mm_ctx* ctx, const void* m, void* dmdt) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_llg_rhs", m, dmdt)) != MM_OK) return s;
  if (m == dmdt) return fail(ctx, MM_ERR_INVALID_ARG, "mm_llg_rhs: dmdt must not alias m");
  if ((s = need_ready(ctx, "mm_llg_rhs", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  return dispatch_eval(ctx, PW_RHS, ctx->terms, m, dmdt);
}

mm_status mm_rk_step(mm_ctx* ctx, void* m_inout, double dt) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_rk_step", m_inout, m_inout)) != MM_OK) return s;
  if (!(dt > 0)) return fail(ctx, MM_ERR_INVALID_ARG, "mm_rk_step: dt must be positive");
  if ((s = need_ready(ctx, "mm_rk_step", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  return ctx->dtype == MM_F32 ? rk_t<float>(ctx, m_inout, dt) : rk_t<double>(ctx, m_inout, dt);
}

// Captures `steps` RK4 steps on m into an executable graph (on a stream of the library's own: the legacy
// default stream cannot be captured).
static mm_status rk_capture(mm_ctx* ctx, void* m, double dt, int steps) {
  if (ctx->rk_graph) { cudaGraphExecDestroy(ctx->rk_graph); ctx->rk_graph = nullptr; }
  cudaError_t e = cudaSuccess;
  if (!ctx->rk_capture_stream) e = cudaStreamCreateWithFlags(&ctx->rk_capture_stream, cudaStreamNonBlocking);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_rk_steps: stream", e);
  cudaStream_t user = ctx->stream;
  const unsigned long long l0 = ctx->launches;
  ctx->stream = ctx->rk_capture_stream;
  e = cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal);
  mm_status s = e == cudaSuccess ? MM_OK : cuda_fail(ctx, "mm_rk_steps: begin capture", e);
  for (int i = 0; i < steps && s == MM_OK; ++i)
    s = ctx->dtype == MM_F32 ? rk_t<float>(ctx, m, dt) : rk_t<double>(ctx, m, dt);
  cudaGraph_t graph = nullptr;
  if (e == cudaSuccess) {
    const cudaError_t e2 = cudaStreamEndCapture(ctx->stream, &graph);
    if (s == MM_OK && e2 != cudaSuccess) s = cuda_fail(ctx, "mm_rk_steps: end capture", e2);
  }
  ctx->stream = user;
  ctx->rk_graph_launches = ctx->launches - l0;   // kernels one replay enqueues
  ctx->launches = l0;
  if (s == MM_OK) {
    e = cudaGraphInstantiate(&ctx->rk_graph, graph, 0);
    if (e != cudaSuccess) s = cuda_fail(ctx, "mm_rk_steps: instantiate", e);
  }
  if (graph) cudaGraphDestroy(graph);
  if (s != MM_OK) { ctx->rk_graph = nullptr; return s; }
  ctx->rk_graph_m = m; ctx->rk_graph_dt = dt; ctx->rk_graph_steps = steps; ctx->rk_graph_epoch = ctx->epoch;
  return MM_OK;
}

mm_status mm_rk_steps(mm_ctx* ctx, void* m_inout, double dt, int n_steps) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_rk_steps", m_inout, m_inout)) != MM_OK) return s;
  if (!(dt > 0) || n_steps < 0) return fail(ctx, MM_ERR_INVALID_ARG, "mm_rk_steps: need dt > 0 and n_steps >= 0");
  if ((s = need_ready(ctx, "mm_rk_steps", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  constexpr int kChunk = 128;
  int left = n_steps;
  if (ctx->prof.on) {   // per-kernel events cannot be recorded from a graph: plain launches
    for (; left > 0 && s == MM_OK; --left) s = mm_rk_step(ctx, m_inout, dt);
    return s;
  }
  while (left > 0) {
    const int chunk = left < kChunk ? left : kChunk;
    const bool have = ctx->rk_graph && ctx->rk_graph_m == m_inout && ctx->rk_graph_dt == dt &&
                      ctx->rk_graph_steps == chunk && ctx->rk_graph_epoch == ctx->epoch;
    // a short tail that would evict a cached full chunk runs as plain steps instead
    if (!have && chunk < kChunk && ctx->rk_graph && ctx->rk_graph_steps == kChunk && chunk < 16) {
      for (; left > 0 && s == MM_OK; --left) s = mm_rk_step(ctx, m_inout, dt);
      return s;
    }
    if (!have && (s = rk_capture(ctx, m_inout, dt, chunk)) != MM_OK) return s;
    const cudaError_t e = cudaGraphLaunch(ctx->rk_graph, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "mm_rk_steps: graph launch", e);
    ctx->launches += ctx->rk_graph_launches;
    left -= chunk;
  }
  return MM_OK;
}

}  // extern "C"

// ---- Barzilai-Borwein minimiser iteration (bb.cu)

template <typename T> static mm_status bb_step_t(mm_ctx* c, void* m) {
  const size_t n3 = (size_t)c->nx * c->ny * c->nz * 3;
  const size_t pitch = align256(n3 * c->es) / c->es;       // the RKF45 stage buffers, reused (never both at once)
  T* K = reinterpret_cast<T*>(c->scr + c->off_rkf);
  T* g = K, *gp = K + pitch, *mp = K + 2 * pitch;
  mm_status s = eval_t<T>(c, PW_MIN_G, m, g, nullptr, pw_of<T>(c, c->terms));
  if (s != MM_OK) return s;
  cudaError_t e = bb_iterate_launch<T>(reinterpret_cast<BbState*>(c->pers + c->off_bbstate), static_cast<T*>(m), g,
                                       mp, gp, reinterpret_cast<double*>(c->pers + c->off_bbpart), n3, c->stream,
                                       &c->launches);
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "mm_minimize_step", e);
}

// ---- adaptive RKF45 (rkf45.cu)

template <typename T> static mm_status rkf_step_t(mm_ctx* c, void* m) {
  const size_t n3 = (size_t)c->nx * c->ny * c->nz * 3;
  // K_1..K_6 contiguous, n3 reals apart; the stage state and the 5th-order candidate reuse the RK4 buffers
  T* K = reinterpret_cast<T*>(c->scr + c->off_rkf);
  RkfState* sd = reinterpret_cast<RkfState*>(c->pers + c->off_rkstate);
  T* stage = reinterpret_cast<T*>(c->scr + c->off_msa);
  T* cand = reinterpret_cast<T*>(c->scr + c->off_msb);
  const PwParams<T> p = pw_of<T>(c, c->terms);
  mm_status s = eval_t<T>(c, PW_RHS, m, K, nullptr, p);
  for (int i = 1; i <= 5 && s == MM_OK; ++i) {
    cudaError_t e = rkf_combine_launch<T>(sd, static_cast<const T*>(m), K, n3, i, rkf_row(i), stage, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, "mm_rkf45_step: stage combination", e);
    ++c->launches;
    s = eval_t<T>(c, PW_RHS, stage, K + (size_t)i * n3, nullptr, p);
  }
  if (s != MM_OK) return s;
  cudaError_t e = rkf_finish_launch<T>(sd, static_cast<T*>(m), K, n3, cand, c->stream, &c->launches);
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "mm_rkf45_step: finish", e);
}

extern "C" {

mm_status mm_rkf45_init(mm_ctx* ctx, double t0, double dt0, double tol, double dt_min, double dt_max) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->pers) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_rkf45_init: mm_ctx_set_workspace not called");
  if (!(dt0 > 0) || !(tol > 0) || dt_min < 0 || !(dt_max >= dt_min) || dt0 < dt_min || dt0 > dt_max)
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_rkf45_init: need tol > 0 and 0 <= dt_min <= dt0 <= dt_max, dt0 > 0");
  RkfState& h = ctx->rk_host;
  h = RkfState{};
  h.t = t0; h.dt = dt0; h.tol = tol; h.dt_min = dt_min; h.dt_max = dt_max;
  cudaError_t e = cudaMemcpyAsync(ctx->pers + ctx->off_rkstate, &h, sizeof(RkfState), cudaMemcpyHostToDevice,
                                  ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_rkf45_init", e);
  ctx->rk_ready = true;
  return MM_OK;
}

mm_status mm_rkf45_step(mm_ctx* ctx, void* m_inout) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_rkf45_step", m_inout, m_inout)) != MM_OK) return s;
  if ((s = need_ready(ctx, "mm_rkf45_step", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  if (!ctx->rk_ready) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_rkf45_step: mm_rkf45_init not called");
  return ctx->dtype == MM_F32 ? rkf_step_t<float>(ctx, m_inout) : rkf_step_t<double>(ctx, m_inout);
}

mm_status mm_rkf45_state(mm_ctx* ctx, double* t, double* dt_next, double* err_last, double* dt_last,
                         int* accepted_last, unsigned long long* n_accepted, unsigned long long* n_rejected) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->rk_ready) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_rkf45_state: mm_rkf45_init not called");
  RkfState h;
  cudaError_t e = cudaMemcpyAsync(&h, ctx->pers + ctx->off_rkstate, sizeof(RkfState), cudaMemcpyDeviceToHost,
                                  ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_rkf45_state", e);
  if (t) *t = h.t;
  if (dt_next) *dt_next = h.dt;
  if (err_last) *err_last = h.err;
  if (dt_last) *dt_last = h.dt_last;
  if (accepted_last) *accepted_last = h.accept;
  if (n_accepted) *n_accepted = h.n_acc;
  if (n_rejected) *n_rejected = h.n_rej;
  return MM_OK;
}

// ---- Barzilai-Borwein minimiser (bb.cu)

mm_status mm_minimize_init(mm_ctx* ctx, double tau0, double tau_min, double tau_max, double tol) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->pers) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_minimize_init: mm_ctx_set_workspace not called");
  if (!(tau0 > 0) || tau_min < 0 || !(tau_max >= tau_min) || tol < 0 || !std::isfinite(tau0) || !std::isfinite(tau_max))
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_minimize_init: need tau0 > 0, 0 <= tau_min <= tau_max, tol >= 0");
  BbState h{};
  h.tau0 = tau0; h.tau_min = tau_min; h.tau_max = tau_max; h.tol = tol;
  cudaError_t e = cudaMemcpyAsync(ctx->pers + ctx->off_bbstate, &h, sizeof(BbState), cudaMemcpyHostToDevice,
                                  ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_minimize_init", e);
  ctx->bb_ready = true;
  return MM_OK;
}

mm_status mm_minimize_step(mm_ctx* ctx, void* m_inout) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_minimize_step", m_inout, m_inout)) != MM_OK) return s;
  if ((s = need_ready(ctx, "mm_minimize_step", ctx->terms & MM_TERM_DEMAG)) != MM_OK) return s;
  if (!ctx->bb_ready) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_minimize_step: mm_minimize_init not called");
  return ctx->dtype == MM_F32 ? bb_step_t<float>(ctx, m_inout) : bb_step_t<double>(ctx, m_inout);
}

mm_status mm_minimize_state(mm_ctx* ctx, unsigned long long* iterations, double* tau_last, double* dm_max,
                            int* converged) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!ctx->bb_ready) return fail(ctx, MM_ERR_NOT_INITIALISED, "mm_minimize_state: mm_minimize_init not called");
  BbState h;
  cudaError_t e = cudaMemcpyAsync(&h, ctx->pers + ctx->off_bbstate, sizeof(BbState), cudaMemcpyDeviceToHost,
                                  ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_minimize_state", e);
  if (iterations) *iterations = h.n;
  if (tau_last) *tau_last = h.tau;
  if (dm_max) *dm_max = h.dm_max;
  if (converged) *converged = h.converged;
  return MM_OK;
}

mm_status mm_minimize(mm_ctx* ctx, void* m_inout, int max_iter, int check_every, unsigned long long* iterations,
                      int* converged) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (max_iter < 0 || check_every < 1)
    return fail(ctx, MM_ERR_INVALID_ARG, "mm_minimize: need max_iter >= 0 and check_every >= 1");
  unsigned long long n = 0;
  int conv = 0;
  mm_status s = mm_minimize_state(ctx, &n, nullptr, nullptr, &conv);
  const unsigned long long n0 = n;
  while (s == MM_OK && !conv && n - n0 < (unsigned long long)max_iter) {
    unsigned long long todo = (unsigned long long)max_iter - (n - n0);
    if (todo > (unsigned long long)check_every) todo = check_every;
    for (unsigned long long i = 0; i < todo && s == MM_OK; ++i) s = mm_minimize_step(ctx, m_inout);
    if (s == MM_OK) s = mm_minimize_state(ctx, &n, nullptr, nullptr, &conv);   // the only synchronisation
  }
  if (iterations) *iterations = n;
  if (converged) *converged = conv;
  return s;
}

// ---- mm_demag_field_static: the convolution with its spectra in a static device array (no allocation)

}  // extern "C"

// The spectra A1, A2 of mm_demag_field_static.  One copy per GPU that loads this module, held until exit.
// In host code `g_static_scratch` is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) unsigned char g_static_scratch[MM_STATIC_SCRATCH_BYTES];

constexpr int kMaxStaticDevices = 64;
static unsigned char* g_static_ptr[kMaxStaticDevices] = {nullptr};   // device address of the array, per device ordinal

// device address of g_static_scratch on the current device, looked up once per device
static cudaError_t static_scratch_ptr(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxStaticDevices) return cudaErrorInvalidDevice;
  unsigned char* p = __atomic_load_n(&g_static_ptr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    void* q = nullptr;
    e = cudaGetSymbolAddress(&q, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!q || ((uintptr_t)q & 255)) return cudaErrorInvalidSymbol;
    p = static_cast<unsigned char*>(q);
    __atomic_store_n(&g_static_ptr[dev], p, __ATOMIC_RELEASE);   // every thread finds the same address
  }
  *out = p;
  return cudaSuccess;
}

// bytes of the two spectra (they sit first in the scratch carve-up: off_a1 = 0), or 0 where the path needs more
static size_t static_need(const mm_ctx* c) {
  if (c->ms_cells || c->embed || c->slabs) return 0;
  return c->off_hd;
}

template <typename T> static mm_status demag_static_t(mm_ctx* c, unsigned char* sp, const void* m, void* H) {
  Cx<T>* A1 = reinterpret_cast<Cx<T>*>(sp + c->off_a1);
  Cx<T>* A2 = reinterpret_cast<Cx<T>*>(sp + c->off_a2);
  cudaError_t e;
  if (c->mixed) {
    const MixedPlans pl{c->geom.px, c->geom.py, c->geom.pz};
    MixedBufs<T> b = mixed_bufs_of<T>(c);
    b.A1 = A1; b.A2 = A2;
    e = demag_mixed_launch<T>(c->fgeom, pl, b, static_cast<const T*>(m), static_cast<T*>(H), (T)(-c->Ms), c->stream,
                              &c->launches, &c->prof);
  } else if (c->fast) {
    FastBufs<T> b = fast_bufs_of<T>(c);
    b.A1 = A1; b.A2 = A2;
    e = demag_fast_launch<T>(c->fgeom, b, static_cast<const T*>(m), static_cast<T*>(H), (T)(-c->Ms), c->stream,
                             &c->launches, &c->prof);
  } else {
    DemagBufs<T> b = bufs_of<T>(c);
    b.A1 = A1; b.A2 = A2;
    e = demag_field_launch<T>(c->geom, b, static_cast<const T*>(m), static_cast<T*>(H), (T)(-c->Ms), c->stream,
                              &c->launches, &c->prof);
  }
  return e == cudaSuccess ? MM_OK : cuda_fail(c, "mm_demag_field_static launch", e);
}

extern "C" {

mm_status mm_static_scratch_info(const mm_ctx* ctx, size_t* capacity, size_t* needed) {
  if (capacity) *capacity = MM_STATIC_SCRATCH_BYTES;
  if (ctx && needed) *needed = static_need(ctx);
  unsigned char* sp = nullptr;
  const cudaError_t e = static_scratch_ptr(&sp);
  if (e == cudaSuccess) return MM_OK;
  if (ctx) return cuda_fail(const_cast<mm_ctx*>(ctx), "mm_static_scratch_info: cudaGetSymbolAddress", e);
  snprintf(g_create_error, sizeof g_create_error, "mm_static_scratch_info: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  return MM_ERR_CUDA;
}

mm_status mm_demag_field_static(mm_ctx* ctx, const void* m, void* H) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  mm_status s;
  if ((s = check_ptr(ctx, "mm_demag_field_static", m, H)) != MM_OK) return s;
  if (m == H) return fail(ctx, MM_ERR_INVALID_ARG, "mm_demag_field_static: H must not alias m");
  if ((s = need_ready(ctx, "mm_demag_field_static", true)) != MM_OK) return s;
  const size_t need = static_need(ctx);
  if (need == 0)
    return fail(ctx, MM_ERR_NOT_IMPLEMENTED,
                "mm_demag_field_static: per-cell Ms, embedded meshes and slabs need more than the spectra; use mm_demag_field");
  if (need > (size_t)MM_STATIC_SCRATCH_BYTES)
    return fail(ctx, MM_ERR_WORKSPACE,
                "mm_demag_field_static: the spectra of this mesh need %zu bytes, the static array holds %zu; use mm_demag_field",
                need, (size_t)MM_STATIC_SCRATCH_BYTES);
  unsigned char* sp = nullptr;
  const cudaError_t e = static_scratch_ptr(&sp);
  if (e != cudaSuccess) return cuda_fail(ctx, "mm_demag_field_static: cudaGetSymbolAddress", e);
  return ctx->dtype == MM_F32 ? demag_static_t<float>(ctx, sp, m, H) : demag_static_t<double>(ctx, sp, m, H);
}

// ---- host-buffer variants: H2D, device path, D2H, synchronise

static mm_status host_call(mm_ctx* ctx, const char* fn, int which, const void* in_host, void* out_host,
                           double dt) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (!in_host || !out_host) return fail(ctx, MM_ERR_INVALID_ARG, "%s: NULL host pointer", fn);
  if (!ctx->scr) return fail(ctx, MM_ERR_NOT_INITIALISED, "%s: mm_ctx_set_workspace not called", fn);
  const size_t n3 = (size_t)ctx->nx * ctx->ny * ctx->nz * 3 * ctx->es;
  void* din = ctx->scr + ctx->off_sin;
  void* dout = ctx->scr + ctx->off_sout;
  cudaError_t e = cudaMemcpyAsync(din, in_host, n3, cudaMemcpyHostToDevice, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, fn, e);
  mm_status s;
  switch (which) {
    case 0: s = mm_demag_field(ctx, din, dout); break;
    case 1: s = mm_heff(ctx, din, dout); break;
    case 2: s = mm_llg_rhs(ctx, din, dout); break;
    default: s = mm_rk_step(ctx, din, dt); dout = din; break;
  }
  if (s != MM_OK) return s;
  e = cudaMemcpyAsync(out_host, dout, n3, cudaMemcpyDeviceToHost, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, fn, e);
  e = cudaStreamSynchronize(ctx->stream);
  return e == cudaSuccess ? MM_OK : cuda_fail(ctx, fn, e);
}

mm_status mm_demag_field_host(mm_ctx* ctx, const void* m_host, void* H_host) {
  return host_call(ctx, "mm_demag_field_host", 0, m_host, H_host, 0);
}
mm_status mm_heff_host(mm_ctx* ctx, const void* m_host, void* H_host) {
  return host_call(ctx, "mm_heff_host", 1, m_host, H_host, 0);
}
mm_status mm_llg_rhs_host(mm_ctx* ctx, const void* m_host, void* dmdt_host) {
  return host_call(ctx, "mm_llg_rhs_host", 2, m_host, dmdt_host, 0);
}
mm_status mm_rk_step_host(mm_ctx* ctx, void* m_inout_host, double dt) {
  return host_call(ctx, "mm_rk_step_host", 3, m_inout_host, m_inout_host, dt);
}

// count independent evaluations: the upload of state i + 1 and the download of result i - 1 run on copy streams
// of their own beside the kernels of state i, two staging slots per direction (slot 1 = the RK4 stage buffers).
static mm_status host_batch(mm_ctx* ctx, const char* fn, int which, const void* const* m_host, void* const* dmdt_host,
                            int count) {
  if (!ctx) return MM_ERR_INVALID_ARG;
  if (count < 0 || (count > 0 && (!m_host || !dmdt_host))) return fail(ctx, MM_ERR_INVALID_ARG, "%s: NULL array or negative count", fn);
  for (int i = 0; i < count; ++i)
    if (!m_host[i] || !dmdt_host[i]) return fail(ctx, MM_ERR_INVALID_ARG, "%s: NULL host pointer at index %d", fn, i);
  mm_status s;
  if ((s = need_ready(ctx, fn, which == 0 || (ctx->terms & MM_TERM_DEMAG) != 0)) != MM_OK) return s;
  if (count == 0) return MM_OK;
  cudaError_t e = cudaSuccess;
  if (!ctx->h2d_stream) {   // streams and events hold no device memory
    if ((e = cudaStreamCreateWithFlags(&ctx->h2d_stream, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(ctx, fn, e);
    if ((e = cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(ctx, fn, e);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
      e = cudaEventCreateWithFlags(&ctx->ev_in[i], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_comp[i], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_out[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, fn, e);
  }
  const size_t n3 = (size_t)ctx->nx * ctx->ny * ctx->nz * 3 * ctx->es;
  void* din[2] = {ctx->scr + ctx->off_sin, ctx->scr + ctx->off_msa};
  void* dout[2] = {ctx->scr + ctx->off_sout, ctx->scr + ctx->off_msb};
  // earlier work on the context's stream may still use the slots
  if ((e = cudaStreamSynchronize(ctx->stream)) != cudaSuccess) return cuda_fail(ctx, fn, e);
  for (int i = 0; i < count; ++i) {
    const int k = i & 1;
    if (i >= 2) e = cudaStreamWaitEvent(ctx->h2d_stream, ctx->ev_comp[k], 0);   // evaluation i - 2 has read slot k
    if (e == cudaSuccess) e = cudaMemcpyAsync(din[k], m_host[i], n3, cudaMemcpyHostToDevice, ctx->h2d_stream);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_in[k], ctx->h2d_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->stream, ctx->ev_in[k], 0);
    if (e == cudaSuccess && i >= 2) e = cudaStreamWaitEvent(ctx->stream, ctx->ev_out[k], 0);   // result i - 2 has left slot k
    if (e != cudaSuccess) break;
    s = which == 0 ? mm_demag_field(ctx, din[k], dout[k]) : which == 1 ? mm_heff(ctx, din[k], dout[k]) : mm_llg_rhs(ctx, din[k], dout[k]);
    if (s != MM_OK) {
      cudaStreamSynchronize(ctx->h2d_stream); cudaStreamSynchronize(ctx->stream); cudaStreamSynchronize(ctx->d2h_stream);
      return s;
    }
    e = cudaEventRecord(ctx->ev_comp[k], ctx->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->d2h_stream, ctx->ev_comp[k], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dmdt_host[i], dout[k], n3, cudaMemcpyDeviceToHost, ctx->d2h_stream);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_out[k], ctx->d2h_stream);
    if (e != cudaSuccess) break;
  }
  const cudaError_t e1 = cudaStreamSynchronize(ctx->h2d_stream), e2 = cudaStreamSynchronize(ctx->stream),
                    e3 = cudaStreamSynchronize(ctx->d2h_stream);
  if (e == cudaSuccess) e = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
  return e == cudaSuccess ? MM_OK : cuda_fail(ctx, fn, e);
}

mm_status mm_demag_field_host_batch(mm_ctx* ctx, const void* const* m_host, void* const* H_host, int count) {
  return host_batch(ctx, "mm_demag_field_host_batch", 0, m_host, H_host, count);
}
mm_status mm_heff_host_batch(mm_ctx* ctx, const void* const* m_host, void* const* H_host, int count) {
  return host_batch(ctx, "mm_heff_host_batch", 1, m_host, H_host, count);
}
mm_status mm_llg_rhs_host_batch(mm_ctx* ctx, const void* const* m_host, void* const* dmdt_host, int count) {
  return host_batch(ctx, "mm_llg_rhs_host_batch", 2, m_host, dmdt_host, count);
}

}  // extern "C"
