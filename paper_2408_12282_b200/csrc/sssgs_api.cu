// Host side of libsssgs: context, argument validation, workspace carving, MLP plan, and the
// orchestration of one sssgs_render call (hot-path step a9: geometry once per camera, MLP +
// light channels + shading per light batch; PAPER.md L301 OLAT sweeps).  No CPU fallback exists:
// every step of the path runs in the kernels of this directory.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "internal.cuh"

using namespace sssgs;

struct sssgs_ctx {
  sssgs_config cfg;
  int num_sms = 0;
  int max_lb = 8;
  uint8_t* ws = nullptr;       // workspace base
  bool owns_ws = false;
  size_t ws_bytes = 0;
  // carved pointers
  float4* attr = nullptr;
  GeomBuffers gb{};
  uint8_t* control = nullptr;  // zeroed once per camera
  size_t control_bytes = 0;
  uint32_t* status_depth[4] = {};
  uint32_t* status_tile[2] = {};
  uint32_t* status_emit = nullptr;
  float4* mlp_out[2] = {};     // double-buffered: the MLP of batch k+1 overlaps the raster of batch k
  cudaStream_t side = nullptr; // the MLP runs here, concurrently with the geometry stages
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_mlp[2] = {}, ev_raster[2] = {}, ev_mask = nullptr;
  // sssgs_render_host: the arrays the geometry chain does not need are uploaded on `copy`; the
  // next sssgs_render makes its MLP / attribute work (or, without overlap, everything) wait for them
  cudaStream_t copy = nullptr;
  cudaEvent_t ev_upload = nullptr;
  bool upload_pending = false;
  WeightCache wc{};             // weight cache of a sweep (pool sized from max_instances)
  uint8_t* contrib = nullptr;   // [n] visibility pre-pass flags (inside the control block)
  uint32_t* rows = nullptr;     // [n] Gaussians kept by the pre-pass
  uint8_t* mlp_blob = nullptr;
  uint8_t* bwd_blob = nullptr;
  int64_t launches = 0;
  // optional per-stage timing
  bool profile = false;
  struct Span { int stage; cudaEvent_t a, b; };
  std::vector<Span> spans;        // spans of the last call
  std::vector<cudaEvent_t> pool;  // recycled events
  int stage_launches[SSSGS_NSTAGES] = {};
  // device staging of sssgs_render_host (grown on demand, owned)
  std::vector<std::pair<void*, size_t>> staging;
  std::string err;
};

namespace {

std::string g_create_err;

constexpr size_t kMaxBlobBytes = 512 * 1024;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int fail(sssgs_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf; else g_create_err = buf;
  return code;
}

bool config_ok(const sssgs_config* cfg) {
  if (!cfg) return false;
  if (cfg->max_gaussians < 0 || cfg->max_gaussians > (int64_t)1 << 30) return false;
  if (cfg->max_width <= 0 || cfg->max_height <= 0) return false;
  if (cfg->max_width > 65535 * kTile || cfg->max_height > 65535 * kTile) return false;
  const int64_t tiles = (int64_t)((cfg->max_width + kTile - 1) / kTile) * ((cfg->max_height + kTile - 1) / kTile);
  if (tiles > 65536) return false;  // tile ids are sorted with at most two 8-bit digits
  if (cfg->max_instances < 0 || cfg->max_instances >= (int64_t)1 << 30) return false;
  const int lb = cfg->max_lights_per_pass;
  if (!(lb == 0 || lb == 1 || lb == 4 || lb == 8)) return false;
  if (cfg->flags != 0) return false;
  return true;
}

// Carves the workspace; with base == nullptr only computes the size.
size_t carve(sssgs_ctx* c, const sssgs_config& cfg, uint8_t* base) {
  size_t off = 0;
  auto take = [&](size_t bytes) -> uint8_t* {
    uint8_t* p = base ? base + off : nullptr;
    off += align_up(bytes ? bytes : 16, 256);
    return p;
  };
  const size_t n = (size_t)cfg.max_gaussians, cap = (size_t)cfg.max_instances;
  const size_t tiles = (size_t)((cfg.max_width + kTile - 1) / kTile) * ((cfg.max_height + kTile - 1) / kTile);
  const int lb = cfg.max_lights_per_pass ? cfg.max_lights_per_pass : 8;
  uint8_t* p;
  p = take(n * 48); if (c) c->attr = (float4*)p;
  p = take(n * 16); if (c) c->gb.rec_a = (float4*)p;
  p = take(n * 16); if (c) c->gb.rec_b = (float4*)p;
  p = take(n * 8);  if (c) c->gb.rect = (uint2*)p;
  p = take(n * 4);  if (c) c->gb.touched = (uint32_t*)p;
  for (int k = 0; k < 2; ++k) { p = take(n * 4); if (c) c->gb.dkeys[k] = (uint32_t*)p; }
  for (int k = 0; k < 2; ++k) { p = take(n * 4); if (c) c->gb.dvals[k] = (uint32_t*)p; }
  for (int k = 0; k < 2; ++k) { p = take(cap * 4); if (c) c->gb.ikeys[k] = (uint32_t*)p; }
  for (int k = 0; k < 2; ++k) { p = take(cap * 4); if (c) c->gb.ivals[k] = (uint32_t*)p; }
  p = take(tiles * 8); if (c) c->gb.ranges = (uint2*)p;
  p = take(tiles * 4); if (c) c->gb.tile_order = (uint32_t*)p;
  p = take((tiles + 1) * 4); if (c) c->gb.tile_slot = (uint32_t*)p;
  for (int k = 0; k < 2; ++k) { p = take(n * (size_t)lb * 16); if (c) c->mlp_out[k] = (float4*)p; }
  p = take(n * 4); if (c) c->rows = (uint32_t*)p;
  {  // weight cache: the blended (block, entry) pairs of a view; half an entry per tile instance
     // covers the scenes measured so far (0.13-0.5); beyond that the sweep falls back to the list walks
    size_t chunks = (cap / 2 + 65536) / kWcChunk;
    if (const char* e = getenv("SSSGS_WC_CHUNKS")) chunks = (size_t)atoll(e);  // tuning / test aid
    const size_t npix = (size_t)cfg.max_width * cfg.max_height;
    p = take(tiles * 8 * 4); if (c) c->wc.head = (uint32_t*)p;
    p = take(tiles * 8 * 4); if (c) c->wc.count = (uint32_t*)p;
    p = take(chunks * 4); if (c) c->wc.next = (uint32_t*)p;
    p = take(chunks * kWcChunk * 8); if (c) c->wc.hdr = (uint2*)p;
    p = take(chunks * kWcChunk * 32 * 4); if (c) c->wc.weights = (float*)p;
    p = take(npix * 4); if (c) c->wc.T = (float*)p;
    p = take(npix * 48); if (c) c->wc.gsum = (float4*)p;
    if (c) c->wc.capacity = (uint32_t)chunks;
  }
  p = take(kMaxBlobBytes); if (c) c->mlp_blob = p;
  p = take(kBwdBlobBytes); if (c) c->bwd_blob = p;   // packed weights of the tensor-core MLP backward
  // control block: everything that must be zero at the start of a camera
  const size_t ctrl_begin = off;
  if (c) c->control = base ? base + off : nullptr;
  p = take(6 * 256 * 4); if (c) c->gb.hist = (uint32_t*)p;
  p = take(DC_WORDS * 4); if (c) c->gb.counters = (uint32_t*)p;
  const size_t nblk_d = sort_status_rows((uint32_t)n), nblk_i = sort_status_rows((uint32_t)cap);
  for (int k = 0; k < 4; ++k) { p = take(nblk_d * kRadixMax * 4); if (c) c->status_depth[k] = (uint32_t*)p; }
  for (int k = 0; k < 2; ++k) { p = take(nblk_i * kRadixMax * 4); if (c) c->status_tile[k] = (uint32_t*)p; }
  p = take(((n + kEmitChunk - 1) / kEmitChunk) * 4); if (c) c->status_emit = (uint32_t*)p;
  p = take(n); if (c) c->contrib = p;
  if (c) c->control_bytes = off - ctrl_begin;
  return off;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

// Makes the context's device current for the duration of an ABI call and restores the caller's.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    if (prev == dev) prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// Builds the tensor-core stage list of the MLP.
int build_plan(sssgs_ctx* c, const sssgs_mlp& m, int feat_dim, MlpPlan* plan) {
  if (m.in_dim != 40 + feat_dim) return fail(c, SSSGS_EINVAL, "mlp.in_dim %d != 40 + feat_dim %d", m.in_dim, feat_dim);
  if (m.n_trunk < 1 || m.n_trunk > SSSGS_MAX_TRUNK) return fail(c, SSSGS_EINVAL, "mlp.n_trunk out of range");
  if (m.n_inc_hidden < 0 || m.n_inc_hidden > SSSGS_MAX_INC_HIDDEN) return fail(c, SSSGS_EINVAL, "mlp.n_inc_hidden out of range");
  if (m.activation != SSSGS_ACT_RELU && m.activation != SSSGS_ACT_LEAKY_RELU) return fail(c, SSSGS_EINVAL, "mlp.activation");
  if (m.dtype != SSSGS_F32 && m.dtype != SSSGS_BF16) return fail(c, SSSGS_EINVAL, "mlp.dtype");
  if (m.compute != SSSGS_COMPUTE_FP16 && m.compute != SSSGS_COMPUTE_BF16) return fail(c, SSSGS_EINVAL, "mlp.compute");
  for (int l = 0; l < m.n_trunk; ++l)
    if (m.trunk_width[l] < 16 || m.trunk_width[l] > 128 || m.trunk_width[l] % 16) return fail(c, SSSGS_EINVAL, "trunk width must be a multiple of 16 in [16,128]");
  for (int l = 0; l < m.n_inc_hidden; ++l)
    if (m.inc_hidden_width[l] < 16 || m.inc_hidden_width[l] > 128 || m.inc_hidden_width[l] % 16) return fail(c, SSSGS_EINVAL, "incident hidden width must be a multiple of 16 in [16,128]");
  memset(plan, 0, sizeof *plan);
  plan->in_dim = m.in_dim;
  plan->in_pad = (m.in_dim + 15) / 16 * 16;
  plan->feat_dim = feat_dim;
  plan->activation = m.activation;
  plan->leaky_slope = m.leaky_slope;
  plan->f16 = m.compute == SSSGS_COMPUTE_FP16 ? 1 : 0;
  int off = 0;       // element offset into params
  int d = m.in_dim;  // current un-padded input width
  int ns = 0, w_off = 0, max_kb = 0, max_n = 0;
  auto add = [&](int type, int k, int n_pad, int n_act) -> MlpStage& {
    MlpStage& st = plan->st[ns++];
    st.type = type;
    st.k_pad = (k + 15) / 16 * 16;
    st.n_pad = n_pad;
    st.n_act = n_act;
    st.src_k = k;
    st.w_off = w_off;
    const int kblocks = (st.k_pad + 63) / 64;
    w_off += kblocks * n_pad * 128;
    if (kblocks > max_kb) max_kb = kblocks;
    if (n_pad > max_n) max_n = n_pad;
    st.src_w[0] = st.src_w[1] = st.src_b[0] = st.src_b[1] = 0;
    st.src_rows[0] = st.src_rows[1] = 0;
    return st;
  };
  for (int l = 0; l < m.n_trunk; ++l) {
    const int o = m.trunk_width[l];
    MlpStage& st = add(ST_HIDDEN, d, o, o);
    st.src_w[0] = off; st.src_b[0] = off + o * d; st.src_rows[0] = o;
    off += o * d + o;
    d = o;
  }
  const int sss_w = off, sss_b = off + 3 * d;
  off += 3 * d + 3;
  if (m.n_inc_hidden == 0) {
    MlpStage& st = add(ST_HEAD_JOINT, d, 16, 0);
    st.src_w[0] = sss_w; st.src_b[0] = sss_b; st.src_rows[0] = 3;
    st.src_w[1] = off; st.src_b[1] = off + d; st.src_rows[1] = 1;
    off += d + 1;
  } else {
    int di = d;
    for (int l = 0; l < m.n_inc_hidden; ++l) {
      const int o = m.inc_hidden_width[l];
      if (l == 0) {
        MlpStage& st = add(ST_HEAD_SPLIT_A, di, o + 16, o);
        st.src_w[0] = off; st.src_b[0] = off + o * di; st.src_rows[0] = o;
        st.src_w[1] = sss_w; st.src_b[1] = sss_b; st.src_rows[1] = 3;
      } else {
        MlpStage& st = add(ST_HIDDEN, di, o, o);
        st.src_w[0] = off; st.src_b[0] = off + o * di; st.src_rows[0] = o;
      }
      off += o * di + o;
      di = o;
    }
    MlpStage& st = add(ST_HEAD_SPLIT_B, di, 16, 0);
    st.src_w[0] = off; st.src_b[0] = off + di; st.src_rows[0] = 1;
    off += di + 1;
  }
  plan->n_stages = ns;
  // the biases follow the weights as UMMA operands too (k_mlp.cu: they are added by the tensor core)
  plan->bias_off = (int)align_up((size_t)w_off, 1024);
  plan->blob_bytes = (int)align_up((size_t)plan->bias_off + (size_t)((ns + 3) / 4) * max_n * 128, 1024);
  plan->max_n = max_n;
  plan->max_k_bytes = max_kb * 128 * 128;
  const size_t elem = m.dtype == SSSGS_BF16 ? 2 : 4;
  if (m.params_bytes != (size_t)off * elem)
    return fail(c, SSSGS_EINVAL, "mlp.params_bytes %zu != expected %zu", m.params_bytes, (size_t)off * elem);
  if ((size_t)plan->blob_bytes > kMaxBlobBytes || max_n > 256)
    return fail(c, SSSGS_ECAPACITY, "MLP too large for the context");
  if (mlp_smem_bytes(*plan) > 227 * 1024)
    return fail(c, SSSGS_ECAPACITY, "MLP weights (%d B) + activations do not fit in shared memory", plan->blob_bytes);
  return SSSGS_OK;
}

CamParams make_cam(const sssgs_camera& s) {
  CamParams c;
  memcpy(c.R, s.R, sizeof c.R);
  memcpy(c.t, s.t, sizeof c.t);
  c.fx = s.fx; c.fy = s.fy; c.cx = s.cx; c.cy = s.cy;
  c.tanx = s.tan_half_fovx; c.tany = s.tan_half_fovy;
  c.width = s.width; c.height = s.height; c.znear = s.znear;
  memcpy(c.bg, s.bg, sizeof c.bg);
  for (int k = 0; k < 3; ++k) c.pos[k] = -(s.R[0 + k] * s.t[0] + s.R[3 + k] * s.t[1] + s.R[6 + k] * s.t[2]);
  c.tiles_x = (s.width + kTile - 1) / kTile;
  c.tiles_y = (s.height + kTile - 1) / kTile;
  return c;
}

}  // namespace

extern "C" {

size_t sssgs_workspace_bytes(const sssgs_config* cfg) {
  if (!config_ok(cfg)) return 0;
  return carve(nullptr, *cfg, nullptr);
}

int sssgs_create(const sssgs_config* cfg, sssgs_ctx** out) {
  if (!out) return fail(nullptr, SSSGS_EINVAL, "out is NULL");
  *out = nullptr;
  if (!config_ok(cfg)) return fail(nullptr, SSSGS_EINVAL, "invalid sssgs_config");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev)
    return fail(nullptr, SSSGS_ECUDA, "no CUDA device %d (libsssgs has no CPU fallback)", cfg->device);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) return fail(nullptr, SSSGS_ECUDA, "cudaGetDeviceProperties failed");
  if (prop.major != 10) return fail(nullptr, SSSGS_EARCH, "device is sm_%d%d; libsssgs is built for sm_100a only", prop.major, prop.minor);
  DeviceGuard guard(cfg->device);
  if (!guard.ok) return fail(nullptr, SSSGS_ECUDA, "cudaSetDevice failed");
  sssgs_ctx* c = new (std::nothrow) sssgs_ctx();
  if (!c) return fail(nullptr, SSSGS_ECUDA, "out of host memory");
  c->cfg = *cfg;
  c->num_sms = prop.multiProcessorCount;
  c->max_lb = cfg->max_lights_per_pass ? cfg->max_lights_per_pass : 8;
  c->ws_bytes = carve(nullptr, *cfg, nullptr);
  if (cfg->workspace) {
    if (cfg->workspace_bytes < c->ws_bytes || ((uintptr_t)cfg->workspace & 255u)) {
      delete c;
      return fail(nullptr, SSSGS_EINVAL, "workspace too small or not 256-byte aligned");
    }
    c->ws = (uint8_t*)cfg->workspace;
  } else {
    if (cudaMalloc(&c->ws, c->ws_bytes) != cudaSuccess) {
      delete c;
      return fail(nullptr, SSSGS_ECUDA, "cudaMalloc of %zu workspace bytes failed", c->ws_bytes);
    }
    c->owns_ws = true;
  }
  carve(c, *cfg, c->ws);
  // rows of the MLP output buffers that a sweep skips are still multiplied by zero weights in some
  // rasteriser shapes: they must never hold non-finite bit patterns
  const int lb0 = cfg->max_lights_per_pass ? cfg->max_lights_per_pass : 8;
  if (cfg->max_gaussians > 0 &&
      (cudaMemset(c->mlp_out[0], 0, (size_t)cfg->max_gaussians * lb0 * 16) != cudaSuccess ||
       cudaMemset(c->mlp_out[1], 0, (size_t)cfg->max_gaussians * lb0 * 16) != cudaSuccess)) {
    sssgs_destroy(c);
    return fail(nullptr, SSSGS_ECUDA, "workspace initialisation failed");
  }
  bool ok = cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->copy, cudaStreamNonBlocking) == cudaSuccess;
  cudaEvent_t* evs[] = {&c->ev_fork, &c->ev_join, &c->ev_mlp[0], &c->ev_mlp[1], &c->ev_raster[0], &c->ev_raster[1],
                        &c->ev_mask, &c->ev_upload};
  for (cudaEvent_t* e : evs) ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
  if (!ok) {
    sssgs_destroy(c);
    return fail(nullptr, SSSGS_ECUDA, "could not create the side stream / events");
  }
  *out = c;
  return SSSGS_OK;
}

void sssgs_destroy(sssgs_ctx* c) {
  if (!c) return;
  DeviceGuard guard(c->cfg.device);
  for (auto& s : c->staging)
    if (s.first) cudaFree(s.first);
  for (auto& sp : c->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  for (auto& e : c->pool) cudaEventDestroy(e);
  cudaEvent_t evs[] = {c->ev_fork, c->ev_join, c->ev_mlp[0], c->ev_mlp[1], c->ev_raster[0], c->ev_raster[1], c->ev_mask,
                       c->ev_upload};
  for (cudaEvent_t e : evs)
    if (e) cudaEventDestroy(e);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->copy) cudaStreamDestroy(c->copy);
  if (c->owns_ws && c->ws) cudaFree(c->ws);
  delete c;
}

int sssgs_profile_enable(sssgs_ctx* c, int enable) {
  if (!c) return SSSGS_EINVAL;
  c->profile = enable != 0;
  return SSSGS_OK;
}

int sssgs_profile_read(sssgs_ctx* c, float* stage_ms, int* stage_launches) {
  if (!c || !stage_ms) return SSSGS_EINVAL;
  for (int k = 0; k < SSSGS_NSTAGES; ++k) stage_ms[k] = 0.f;
  for (auto& sp : c->spans) {
    if (cudaEventSynchronize(sp.b) != cudaSuccess) return fail(c, SSSGS_ECUDA, "event sync failed");
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sp.a, sp.b) != cudaSuccess) return fail(c, SSSGS_ECUDA, "event elapsed failed");
    stage_ms[sp.stage] += ms;
  }
  if (stage_launches)
    for (int k = 0; k < SSSGS_NSTAGES; ++k) stage_launches[k] = c->stage_launches[k];
  return SSSGS_OK;
}

// BVH build + ray-traced visibility + SH fit.  The tree lives in workspace regions a
// render rewrites before reading (attribute pack, projection records, MLP outputs, tile rects), so a
// bake needs no memory of its own and leaves nothing a later render depends on.
int sssgs_bake_visibility(sssgs_ctx* c, const sssgs_gaussians* g, const sssgs_bake* b, void* cuda_stream) {
  if (!c) return SSSGS_EINVAL;
  if (!g || !b) return fail(c, SSSGS_EINVAL, "NULL argument");
  if (g->n < 0) return fail(c, SSSGS_EINVAL, "n < 0");
  if (g->n > c->cfg.max_gaussians) return fail(c, SSSGS_ECAPACITY, "n %lld > max_gaussians %lld", (long long)g->n, (long long)c->cfg.max_gaussians);
  if (b->n_dirs < 1 || b->n_dirs > 4096) return fail(c, SSSGS_EINVAL, "n_dirs must be in [1,4096]");
  if (b->sh_degree < 0 || b->sh_degree > 1) return fail(c, SSSGS_EINVAL, "sh_degree must be 0 or 1");
  if (!(b->t_min >= 0.f) || b->t_min > 3.0e38f) return fail(c, SSSGS_EINVAL, "t_min must be finite and >= 0");
  if (!b->dirs || !b->weights || !b->vis_sh_out) return fail(c, SSSGS_EINVAL, "dirs / weights / vis_sh_out is NULL");
  if (!aligned16(b->vis_sh_out)) return fail(c, SSSGS_EINVAL, "vis_sh_out is not 16-byte aligned");
  c->launches = 0;
  if (g->n == 0) return SSSGS_OK;
  if (!g->means || !g->scales || !g->rotations || !g->opacities) return fail(c, SSSGS_EINVAL, "means / scales / rotations / opacities is NULL");
  DeviceGuard guard(c->cfg.device);
  if (!guard.ok) return fail(c, SSSGS_ECUDA, "cudaSetDevice(%d) failed", c->cfg.device);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (c->upload_pending) {  // a preceding sssgs_render_host may still be uploading on the copy stream
    if (cudaStreamWaitEvent(s, c->ev_upload, 0) != cudaSuccess) return fail(c, SSSGS_ECUDA, "stream wait failed");
  }
  const int64_t n = g->n;
  BvhBuffers bb;
  bb.code_of = c->rows;
  bb.sorted_codes = c->gb.dkeys[0];  // free once the codes are sorted (only the index array is read)
  bb.sorted_gid = c->gb.dkeys[1];
  bb.leaf = c->attr;                 // 48 B per Gaussian
  bb.box_lo = c->gb.rec_a;           // rec_a + rec_b are adjacent: 32 B per Gaussian
  bb.box_hi = c->mlp_out[0];         // mlp_out[0] + mlp_out[1] are adjacent: >= 32 B per Gaussian
  bb.parent = (int*)c->gb.rect;      // 8 B per Gaussian
  bb.flags = c->gb.touched;
  uint32_t* cnt = c->gb.counters;
  const int max_blocks = c->num_sms * 4;
  if (cudaMemsetAsync(c->control, 0, c->control_bytes, s) != cudaSuccess ||
      cudaMemsetAsync(bb.flags, 0, (size_t)n * 4, s) != cudaSuccess)
    return fail(c, SSSGS_ECUDA, "memset failed");
  int launches = 0;
  launches += launch_bvh_bounds(n, g->means, cnt + DC_BVH_BOUNDS, max_blocks, s);
  launches += launch_bvh_morton(n, g->means, cnt + DC_BVH_BOUNDS, c->gb.dkeys[0], c->gb.dvals[0], bb.code_of,
                                c->gb.hist, max_blocks, s);
  for (int p = 0; p < 4; ++p)
    launches += launch_depth_pass(c->gb.dkeys, c->gb.dvals, (uint32_t)n, p, c->gb.hist, c->status_depth[p],
                                  cnt + DC_TICKET_BASE + p, cnt + DC_SORT_ERROR, max_blocks, s);
  launches += launch_bvh_build(*g, bb, c->gb.hist, c->gb.dvals[0], c->gb.dvals[1], s);
  launches += launch_bvh_trace(n, bb, b->n_dirs, b->dirs, b->weights, b->t_min, (b->sh_degree + 1) * (b->sh_degree + 1),
                               b->vis_sh_out, b->vis_out, b->positions != 0, c->num_sms, (float4*)c->wc.weights,
                               (size_t)c->wc.capacity * kWcChunk * 32 * 4, s);
  c->launches = launches;
  if (cudaGetLastError() != cudaSuccess) return fail(c, SSSGS_ECUDA, "a bake kernel launch failed");
  return SSSGS_OK;
}

const char* sssgs_last_error(const sssgs_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }
int64_t sssgs_last_launch_count(const sssgs_ctx* c) { return c ? c->launches : 0; }

int sssgs_render(sssgs_ctx* c, const sssgs_gaussians* g, const sssgs_mlp* mlp, const sssgs_camera* cams,
                 int n_cam, const sssgs_light* lights, int n_light, const sssgs_out* out,
                 uint32_t flags, void* cuda_stream) {
  if (!c) return SSSGS_EINVAL;
  if (!g || !mlp || !out || (n_cam > 0 && !cams) || (n_light > 0 && !lights)) return fail(c, SSSGS_EINVAL, "NULL argument");
  if (n_cam < 0 || n_light < 0) return fail(c, SSSGS_EINVAL, "negative count");
  if (flags & ~(uint32_t)(SSSGS_LIGHTS_PER_CAMERA | SSSGS_SUM_LIGHTS | SSSGS_FORWARD_SHADING | SSSGS_TIGHT_LISTS))
    return fail(c, SSSGS_EINVAL, "unknown flags");
  const bool forward = (flags & SSSGS_FORWARD_SHADING) != 0;
  if (forward && ((flags & SSSGS_SUM_LIGHTS) || out->gbuffer || out->aov_diffuse || out->aov_specular))
    return fail(c, SSSGS_EINVAL, "SSSGS_FORWARD_SHADING: no gbuffer / AOV outputs, not with SSSGS_SUM_LIGHTS");
  const bool sum_lights = (flags & SSSGS_SUM_LIGHTS) != 0;
  if (sum_lights && (out->aov_diffuse || out->aov_specular))
    return fail(c, SSSGS_EINVAL, "SSSGS_SUM_LIGHTS: the AOV outputs must be NULL");
  if (g->n < 0) return fail(c, SSSGS_EINVAL, "n < 0");
  if (g->n > c->cfg.max_gaussians) return fail(c, SSSGS_ECAPACITY, "n %lld > max_gaussians %lld", (long long)g->n, (long long)c->cfg.max_gaussians);
  if (g->vis_sh_degree < 0 || g->vis_sh_degree > 1) return fail(c, SSSGS_EINVAL, "vis_sh_degree must be 0 or 1");
  if (g->feat_dim < 0 || g->feat_dim > 88 || g->feat_dim % 4) return fail(c, SSSGS_EINVAL, "feat_dim must be a multiple of 4 in [0,88]");
  if (g->n > 0) {
    const void* req[] = {g->means, g->scales, g->rotations, g->opacities, g->normals, g->base_color,
                         g->roughness, g->metallic, g->subsurface, g->vis_sh};
    for (const void* p : req)
      if (!p || !aligned16(p)) return fail(c, SSSGS_EINVAL, "a Gaussian attribute pointer is NULL or not 16-byte aligned");
    if (g->feat_dim > 0 && (!g->feat || !aligned16(g->feat))) return fail(c, SSSGS_EINVAL, "feat is NULL or misaligned");
  }
  const void* outs[] = {out->rgb, out->gbuffer, out->aov_diffuse, out->aov_specular, out->mlp_out,
                        out->sorted_keys, out->sorted_vals, out->tile_ranges, out->counters};
  for (const void* p : outs)
    if (p && !aligned16(p)) return fail(c, SSSGS_EINVAL, "an output pointer is not 16-byte aligned");
  MlpPlan plan;
  const bool run_mlp = mlp->precomputed_out == nullptr;
  if (run_mlp) {
    if (!mlp->params || !aligned16(mlp->params)) return fail(c, SSSGS_EINVAL, "mlp.params is NULL or misaligned");
    const int rc = build_plan(c, *mlp, g->feat_dim, &plan);
    if (rc != SSSGS_OK) return rc;
  } else if (!aligned16(mlp->precomputed_out)) {
    return fail(c, SSSGS_EINVAL, "mlp.precomputed_out misaligned");
  }
  for (int v = 0; v < n_cam; ++v) {
    const sssgs_camera& cm = cams[v];
    if (cm.width <= 0 || cm.height <= 0) return fail(c, SSSGS_EINVAL, "camera %d: empty image", v);
    if (cm.width > c->cfg.max_width || cm.height > c->cfg.max_height)
      return fail(c, SSSGS_ECAPACITY, "camera %d: %dx%d exceeds the context's %dx%d", v, cm.width, cm.height, c->cfg.max_width, c->cfg.max_height);
    if (!(cm.fx > 0.f) || !(cm.fy > 0.f) || !(cm.znear > 0.f)) return fail(c, SSSGS_EINVAL, "camera %d: fx, fy, znear must be > 0", v);
    // every output is laid out [F][H][W]...: one image size per call
    if (cm.width != cams[0].width || cm.height != cams[0].height)
      return fail(c, SSSGS_EINVAL, "camera %d: %dx%d differs from camera 0 (%dx%d); all cameras of a call must share one image size",
                  v, cm.width, cm.height, cams[0].width, cams[0].height);
  }
  DeviceGuard guard(c->cfg.device);
  if (!guard.ok) return fail(c, SSSGS_ECUDA, "cudaSetDevice(%d) failed", c->cfg.device);

  cudaStream_t s = (cudaStream_t)cuda_stream;
  const uint32_t cap = (uint32_t)c->cfg.max_instances;
  const int max_blocks = c->num_sms * 4;
  int64_t launches = 0;
  int cur_stage = -1;
  auto add = [&](int k) {
    if (k > 0) {
      launches += k;
      if (cur_stage >= 0) c->stage_launches[cur_stage] += k;
    }
    return k;
  };
  auto new_event = [&]() {
    cudaEvent_t e = nullptr;
    if (!c->pool.empty()) { e = c->pool.back(); c->pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
  };
  if (c->profile) {
    for (auto& sp : c->spans) { c->pool.push_back(sp.a); c->pool.push_back(sp.b); }
    c->spans.clear();
  }
  memset(c->stage_launches, 0, sizeof c->stage_launches);
  auto begin = [&](int stage) {
    cur_stage = stage;
    if (c->profile) {
      sssgs_ctx::Span sp{stage, new_event(), new_event()};
      cudaEventRecord(sp.a, s);
      c->spans.push_back(sp);
    }
  };
  auto end = [&]() {
    if (c->profile && !c->spans.empty()) cudaEventRecord(c->spans.back().b, s);
    cur_stage = -1;
  };
  // The MLP depends on the view and the light but not on the geometry stages, so it runs on the
  // context's side stream and overlaps projection / sort / binning (and, in a sweep, the raster of
  // the previous light batch).  With per-stage timing on, everything is serialised on `s` so that
  // each stage is timed alone.
  const bool overlap = run_mlp && !c->profile && g->n > 0 && n_light > 0 && n_cam > 0;
  // MLP work avoidance in light sweeps: which Gaussians are ever blended depends on the view, not
  // on the light.  A visibility pre-pass (the render walk without channels) flags them, and the
  // MLP of every light of that view evaluates the flagged rows only -- the others are never read by
  // a blend, so every output is unchanged.  Worth a pre-pass from 4 lights per view on; off when
  // the caller wants the MLP outputs of all Gaussians.
  const bool use_mask = run_mlp && g->n > 0 && n_light >= 4 && !out->mlp_out;
  cudaStream_t sm = overlap ? c->side : s;
  if (overlap) {
    if (cudaEventRecord(c->ev_fork, s) != cudaSuccess || cudaStreamWaitEvent(sm, c->ev_fork, 0) != cudaSuccess)
      return fail(c, SSSGS_ECUDA, "stream fork failed");
  }

  if (c->upload_pending) {  // set by sssgs_render_host: late uploads gate the MLP / attribute work
    c->upload_pending = false;
    if (cudaStreamWaitEvent(sm, c->ev_upload, 0) != cudaSuccess) return fail(c, SSSGS_ECUDA, "stream wait failed");
  }
  begin(SSSGS_STAGE_PACK);
  if (add(launch_pack_attr(*g, c->attr, sm)) < 0) return fail(c, SSSGS_ECUDA, "launch failed");
  if (run_mlp && g->n > 0 && n_light > 0) add(launch_mlp_pack(*mlp, plan, c->mlp_blob, sm));
  end();
  int64_t batch_no = 0;

  const int64_t npix_max = 0;
  (void)npix_max;
  for (int v = 0; v < n_cam; ++v) {
    const CamParams cam = make_cam(cams[v]);
    const int tiles = cam.tiles_x * cam.tiles_y;
    const int64_t npix = (int64_t)cam.width * cam.height;
    if (cudaMemsetAsync(c->control, 0, c->control_bytes, s) != cudaSuccess) return fail(c, SSSGS_ECUDA, "memset failed");
    uint32_t* cnt = c->gb.counters;
    // ---- a3: projection ------------------------------------------------------------------------
    begin(SSSGS_STAGE_PROJECT);
    add(launch_project(*g, cam, c->gb, (flags & SSSGS_TIGHT_LISTS) ? 1 : 0, s));
    end();
    begin(SSSGS_STAGE_DEPTH_SORT);
    // ---- a5 (1/2): all Gaussians by depth, 4 x 8 bits, stable ------------------------------------
    const uint32_t n32 = (uint32_t)g->n;
    for (int p = 0; p < 4; ++p)
      add(launch_depth_pass(c->gb.dkeys, c->gb.dvals, n32, p, c->gb.hist, c->status_depth[p],
                            cnt + DC_TICKET_BASE + p, cnt + DC_SORT_ERROR, max_blocks, s));
    end();
    // ---- a4: scan + expansion into (tile, Gaussian) instances, in depth order ---------------------
    int tb = 1;
    while ((1 << tb) < tiles) ++tb;
    const int npass = tb > 8 ? 2 : 1;
    const int bits0 = npass == 2 ? (tb + 1) / 2 : tb, bits1 = npass == 2 ? tb - bits0 : 0;
    begin(SSSGS_STAGE_EMIT);
    add(launch_emit(g->n, cam, c->gb, cap, 0, bits0, bits0, bits1, c->status_emit,
                    cnt + DC_TICKET_BASE + 4, s));
    end();
    begin(SSSGS_STAGE_TILE_SORT);
    // ---- a5 (2/2): instances by tile id, stable -> per tile (depth, index) order -------------------
    add(launch_sort_pass(c->gb.ikeys[0], c->gb.ivals[0], c->gb.ikeys[1], c->gb.ivals[1], cnt + DC_INSTANCES,
                         cap, 0, bits0, c->gb.hist + 4 * 256, c->status_tile[0], cnt + DC_TICKET_BASE + 5,
                         cnt + DC_SORT_ERROR, max_blocks, s));
    if (npass == 2)
      add(launch_sort_pass(c->gb.ikeys[1], c->gb.ivals[1], c->gb.ikeys[0], c->gb.ivals[0], cnt + DC_INSTANCES,
                           cap, bits0, bits1, c->gb.hist + 5 * 256, c->status_tile[1],
                           cnt + DC_TICKET_BASE + 6, cnt + DC_SORT_ERROR, max_blocks, s));
    end();
    const int fi = npass & 1;
    const uint32_t* sorted_tiles = c->gb.ikeys[fi];
    const uint32_t* sorted_vals = c->gb.ivals[fi];
    // ---- a6: tile ranges ---------------------------------------------------------------------------
    begin(SSSGS_STAGE_RANGES);
    add(launch_ranges(sorted_tiles, cam, c->gb, cap,
                      out->tile_ranges ? (uint2*)(out->tile_ranges + (size_t)v * tiles * 2) : nullptr,
                      out->counters ? out->counters + (size_t)v * SSSGS_NCOUNTERS : nullptr,
                      run_mlp && g->n > 0 && n_light > 0, s));
    if (out->sorted_keys || out->sorted_vals)
      add(launch_export_lists(sorted_tiles, sorted_vals, c->gb, cap,
                              out->sorted_keys ? out->sorted_keys + (size_t)v * cap : nullptr,
                              out->sorted_vals ? out->sorted_vals + (size_t)v * cap : nullptr, s));
    end();
    // The pre-pass also caches the compositing weights of the view (deferred path): the per-light
    // walks then stream the cache instead of walking the lists again.
    const bool use_cache = use_mask && !forward && c->wc.capacity > 0;
    if (use_mask) {
      c->wc.chunks = cnt + DC_WC_CHUNKS;
      c->wc.overflow = cnt + DC_WC_OVERFLOW;
      begin(SSSGS_STAGE_PREPASS);
      add(launch_mark_contrib(cam, c->gb, sorted_vals, c->contrib, use_cache ? &c->wc : nullptr, s));
      add(launch_compact_contrib(c->contrib, g->n, c->rows, cnt + DC_CONTRIB_ROWS, raster_reads_unblended_rows(tiles),
                                 c->mlp_out[0], c->mlp_out[1], n_light < c->max_lb ? n_light : c->max_lb, s));
      end();
      if (overlap && (cudaEventRecord(c->ev_mask, s) != cudaSuccess || cudaStreamWaitEvent(sm, c->ev_mask, 0) != cudaSuccess))
        return fail(c, SSSGS_ECUDA, "stream wait failed");
    }
    // ---- per light batch: a1+a2 MLP, a7+a8 raster + shade -------------------------------------------
    for (int l0 = 0; l0 < n_light; l0 += c->max_lb) {
      const int nl = n_light - l0 < c->max_lb ? n_light - l0 : c->max_lb;
      LightBatch lb;
      memset(&lb, 0, sizeof lb);
      for (int l = 0; l < nl; ++l) {
        const sssgs_light& L = lights[(flags & SSSGS_LIGHTS_PER_CAMERA) ? (size_t)v * n_light + l0 + l : (size_t)(l0 + l)];
        memcpy(lb.l[l].pos, L.position, 12);
        memcpy(lb.l[l].intensity, L.intensity, 12);
      }
      const int64_t frame0 = (int64_t)v * n_light + l0;
      const int buf = (int)(batch_no & 1);
      float4* mlp_buf = c->mlp_out[buf];
      begin(SSSGS_STAGE_MLP);
      if (run_mlp) {
        // buffer `buf` was last read by the raster of batch_no - 2
        if (overlap && batch_no >= 2 && cudaStreamWaitEvent(sm, c->ev_raster[buf], 0) != cudaSuccess)
          return fail(c, SSSGS_ECUDA, "stream wait failed");
        // The MLP of a camera's first light batch runs next to the geometry chain (side stream).  One MLP
        // CTA fills an SM (512 threads x 128 registers, TMEM), so the two do not share SMs: the MLP is
        // confined to a third of them and the latency-bound geometry kernels keep the rest.  Measured on
        // configs 2 and 4 (profiles/r02_notes.md): the step time is flat from a third of the SMs upwards
        // (cfg 4: 0.812 ms at 49 SMs, 0.806 at 60 ... 148) and rises below it (0.95 at 37, 1.21 at 25).
        int mlp_ctas = c->num_sms;
        if (overlap && l0 == 0 && !use_mask) mlp_ctas = (c->num_sms + 2) / 3;
        const int k = launch_mlp(*g, plan, c->mlp_blob, cam, lb, nl, mlp_buf,
                                 out->mlp_out ? out->mlp_out + frame0 * g->n * 4 : nullptr, g->n * 4,
                                 mlp_ctas, use_mask ? c->rows : nullptr, use_mask ? cnt + DC_CONTRIB_ROWS : nullptr,
                                 out->counters ? out->counters + (size_t)v * SSSGS_NCOUNTERS + SSSGS_CNT_MLP_ROWS : nullptr, sm);
        if (k < 0) return fail(c, SSSGS_ECUDA, "MLP kernel configuration failed: %s", cudaGetErrorString(cudaGetLastError()));
        add(k);
        if (forward) add(launch_shade_gaussians(g->n, nl, g->means, c->attr, cam, lb, mlp_buf, sm));
        if (overlap && (cudaEventRecord(c->ev_mlp[buf], sm) != cudaSuccess || cudaStreamWaitEvent(s, c->ev_mlp[buf], 0) != cudaSuccess))
          return fail(c, SSSGS_ECUDA, "stream join failed");
      } else {
        add(launch_gather_precomputed(mlp->precomputed_out + frame0 * g->n * 4, g->n, nl, g->n * 4, mlp_buf, s));
        if (out->mlp_out && g->n > 0)
          if (cudaMemcpyAsync(out->mlp_out + frame0 * g->n * 4, mlp->precomputed_out + frame0 * g->n * 4,
                              (size_t)nl * g->n * 16, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
            return fail(c, SSSGS_ECUDA, "memcpy failed");
      }
      end();
      begin(SSSGS_STAGE_RASTER);
      if (forward) {
        if (!run_mlp) add(launch_shade_gaussians(g->n, nl, g->means, c->attr, cam, lb, mlp_buf, s));
        add(launch_raster_forward(cam, nl, c->gb, sorted_vals, mlp_buf,
                                  out->rgb ? out->rgb + frame0 * npix * 3 : nullptr, npix, s));
      } else {
      float* o_rgb = out->rgb ? out->rgb + (sum_lights ? (int64_t)v : frame0) * npix * 3 : nullptr;
      float* o_gbuf = out->gbuffer ? out->gbuffer + frame0 * npix * SSSGS_GBUF_CHANNELS : nullptr;
      float* o_ad = out->aov_diffuse ? out->aov_diffuse + frame0 * npix * 3 : nullptr;
      float* o_as = out->aov_specular ? out->aov_specular + frame0 * npix * 3 : nullptr;
      const int smode = sum_lights ? (l0 == 0 ? 1 : 2) : 0;
      if (use_cache) {  // cached walk; the list walk behind it only runs if the cache overflowed
        add(launch_raster_cached(cam, lb, nl, c->gb, c->wc, c->attr, mlp_buf, o_rgb, o_gbuf, o_ad, o_as, npix, smode,
                                 l0 == 0, s));
        add(launch_raster(cam, lb, nl, c->gb, sorted_vals, c->attr, mlp_buf, o_rgb, o_gbuf, o_ad, o_as, npix, smode, s,
                          cnt + DC_WC_OVERFLOW));
      } else
      add(launch_raster(cam, lb, nl, c->gb, sorted_vals, c->attr, mlp_buf,
                        out->rgb ? out->rgb + (sum_lights ? (int64_t)v : frame0) * npix * 3 : nullptr,
                        out->gbuffer ? out->gbuffer + frame0 * npix * SSSGS_GBUF_CHANNELS : nullptr,
                        out->aov_diffuse ? out->aov_diffuse + frame0 * npix * 3 : nullptr,
                        out->aov_specular ? out->aov_specular + frame0 * npix * 3 : nullptr, npix,
                        sum_lights ? (l0 == 0 ? 1 : 2) : 0, s));
      }
      end();
      if (overlap && cudaEventRecord(c->ev_raster[buf], s) != cudaSuccess) return fail(c, SSSGS_ECUDA, "event record failed");
      ++batch_no;
    }
  }
  if (overlap) {  // everything on the side stream is ordered before the end of the call on `s`
    if (cudaEventRecord(c->ev_join, sm) != cudaSuccess || cudaStreamWaitEvent(s, c->ev_join, 0) != cudaSuccess)
      return fail(c, SSSGS_ECUDA, "stream join failed");
  }
  c->launches = launches;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, SSSGS_ECUDA, "CUDA error: %s", cudaGetErrorString(e));
  return SSSGS_OK;
}

// backward of a8 / a7 / a2 for one camera.  Geometry and the MLP forward are run again (they
// are cheap next to the walks), then shading backward per light batch, the back-to-front compositing walk
// and the MLP backward.
int sssgs_render_backward(sssgs_ctx* c, const sssgs_gaussians* g, const sssgs_mlp* mlp, const sssgs_camera* cam_in,
                          const sssgs_light* lights, int n_light, const sssgs_grads* gr, uint32_t flags,
                          void* cuda_stream) {
  if (!c) return SSSGS_EINVAL;
  if (!g || !mlp || !cam_in || !gr || (n_light > 0 && !lights)) return fail(c, SSSGS_EINVAL, "NULL argument");
  if (flags & ~(uint32_t)(SSSGS_TIGHT_LISTS | SSSGS_BACKWARD_FP32))
    return fail(c, SSSGS_EINVAL, "sssgs_render_backward: only SSSGS_TIGHT_LISTS and SSSGS_BACKWARD_FP32 are accepted");
  if (n_light < 0 || g->n < 0) return fail(c, SSSGS_EINVAL, "negative count");
  if (g->n > c->cfg.max_gaussians) return fail(c, SSSGS_ECAPACITY, "n exceeds max_gaussians");
  if (g->vis_sh_degree < 0 || g->vis_sh_degree > 1) return fail(c, SSSGS_EINVAL, "vis_sh_degree must be 0 or 1");
  if (g->feat_dim < 0 || g->feat_dim > 88 || g->feat_dim % 4) return fail(c, SSSGS_EINVAL, "feat_dim must be a multiple of 4 in [0,88]");
  const void* must[] = {gr->grad_opacity, gr->grad_mean2d, gr->grad_conic, gr->grad_depth, gr->grad_attr};
  for (const void* p : must)
    if (!p || !aligned16(p)) return fail(c, SSSGS_EINVAL, "a gradient pointer is NULL or not 16-byte aligned");
  const void* per_light[] = {gr->grad_rgb, gr->gbuffer, gr->grad_gbuffer, gr->grad_mlp_out};
  for (const void* p : per_light)   // per-light arrays are empty without lights
    if (n_light > 0 && (!p || !aligned16(p))) return fail(c, SSSGS_EINVAL, "a per-light gradient pointer is NULL or not 16-byte aligned");
  if (gr->grad_params && !aligned16(gr->grad_params)) return fail(c, SSSGS_EINVAL, "grad_params misaligned");
  if (gr->grad_gbuffer_in && !aligned16(gr->grad_gbuffer_in)) return fail(c, SSSGS_EINVAL, "grad_gbuffer_in misaligned");
  if (gr->grad_gbuffer_in && gr->grad_gbuffer_in == gr->grad_gbuffer)
    return fail(c, SSSGS_EINVAL, "grad_gbuffer_in must not alias grad_gbuffer");
  if (gr->counters && !aligned16(gr->counters)) return fail(c, SSSGS_EINVAL, "counters misaligned");
  const int n_geo = (gr->grad_means ? 1 : 0) + (gr->grad_scales ? 1 : 0) + (gr->grad_rotations ? 1 : 0);
  if (n_geo != 0 && n_geo != 3) return fail(c, SSSGS_EINVAL, "grad_means, grad_scales and grad_rotations: all three or none");
  if (n_geo == 3 && (!aligned16(gr->grad_means) || !aligned16(gr->grad_scales) || !aligned16(gr->grad_rotations)))
    return fail(c, SSSGS_EINVAL, "grad_means / grad_scales / grad_rotations misaligned");
  const int n_in = (gr->grad_feat ? 1 : 0) + (gr->grad_vis_sh ? 1 : 0);
  if (n_in == 1) return fail(c, SSSGS_EINVAL, "grad_feat and grad_vis_sh: both or none");
  if (n_in == 2 && (n_geo != 3 || !gr->grad_params || mlp->precomputed_out || !aligned16(gr->grad_feat) || !aligned16(gr->grad_vis_sh)))
    return fail(c, SSSGS_EINVAL, "grad_feat / grad_vis_sh need grad_means, grad_scales, grad_rotations, grad_params and the MLP (no precomputed_out), 16-byte aligned");
  if (g->n > 0) {
    const void* req[] = {g->means, g->scales, g->rotations, g->opacities, g->normals, g->base_color,
                         g->roughness, g->metallic, g->subsurface, g->vis_sh};
    for (const void* p : req)
      if (!p || !aligned16(p)) return fail(c, SSSGS_EINVAL, "a Gaussian attribute pointer is NULL or not 16-byte aligned");
    if (g->feat_dim > 0 && (!g->feat || !aligned16(g->feat))) return fail(c, SSSGS_EINVAL, "feat is NULL or misaligned");
  }
  const sssgs_camera& cm = *cam_in;
  if (cm.width <= 0 || cm.height <= 0 || cm.width > c->cfg.max_width || cm.height > c->cfg.max_height)
    return fail(c, SSSGS_ECAPACITY, "camera size out of range");
  if (!(cm.fx > 0.f) || !(cm.fy > 0.f) || !(cm.znear > 0.f)) return fail(c, SSSGS_EINVAL, "fx, fy, znear must be > 0");
  MlpPlan plan;
  const bool run_mlp = mlp->precomputed_out == nullptr;
  if (run_mlp) {
    if (!mlp->params || !aligned16(mlp->params)) return fail(c, SSSGS_EINVAL, "mlp.params is NULL or misaligned");
    if (mlp->dtype != SSSGS_F32) return fail(c, SSSGS_EINVAL, "sssgs_render_backward needs fp32 parameters (mlp.dtype = SSSGS_F32)");
    const int rc = build_plan(c, *mlp, g->feat_dim, &plan);
    if (rc != SSSGS_OK) return rc;
  }
  DeviceGuard guard(c->cfg.device);
  if (!guard.ok) return fail(c, SSSGS_ECUDA, "cudaSetDevice(%d) failed", c->cfg.device);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (c->upload_pending) {
    c->upload_pending = false;
    if (cudaStreamWaitEvent(s, c->ev_upload, 0) != cudaSuccess) return fail(c, SSSGS_ECUDA, "stream wait failed");
  }
  const int64_t n = g->n;
  const CamParams cam = make_cam(cm);
  const int tiles = cam.tiles_x * cam.tiles_y;
  const int64_t npix = (int64_t)cam.width * cam.height;
  const uint32_t cap = (uint32_t)c->cfg.max_instances;
  const int max_blocks = c->num_sms * 4;
  int64_t launches = 0;
  // every output starts from zero (the walks accumulate with atomics)
  launches += launch_zero(gr->grad_mlp_out, (int64_t)n_light * n * 4, s);
  launches += launch_zero(gr->grad_opacity, n, s);
  launches += launch_zero(gr->grad_mean2d, n * 2, s);
  launches += launch_zero(gr->grad_conic, n * 3, s);
  launches += launch_zero(gr->grad_depth, n, s);
  launches += launch_zero(gr->grad_attr, n * 9, s);
  if (gr->grad_params) launches += launch_zero(gr->grad_params, (int64_t)(mlp->params_bytes / 4), s);
  // grad_gbuffer is written in full by the shading backward of every light batch; only the degenerate call
  // (no Gaussians: nothing below runs) has to clear it here
  if (n == 0) launches += launch_zero(gr->grad_gbuffer, (int64_t)n_light * npix * 16, s);
  if (n_geo == 3) {   // the a1 backward accumulates into these, the projection backward adds to them
    launches += launch_zero(gr->grad_means, n * 3, s);
    launches += launch_zero(gr->grad_scales, n * 3, s);
    launches += launch_zero(gr->grad_rotations, n * 4, s);
  }
  const int ncoef = (g->vis_sh_degree + 1) * (g->vis_sh_degree + 1);
  if (n_in == 2) {
    launches += launch_zero(gr->grad_feat, n * g->feat_dim, s);
    launches += launch_zero(gr->grad_vis_sh, n * ncoef, s);
  }
  if (n == 0 || n_light == 0) {
    if (gr->counters && cudaMemsetAsync(gr->counters, 0, SSSGS_NCOUNTERS * sizeof(int64_t), s) != cudaSuccess)
      return fail(c, SSSGS_ECUDA, "memset failed");
    c->launches = launches;
    return SSSGS_OK;
  }
  // ---- forward state: attributes, geometry of the camera (as sssgs_render) -------------------------
  launches += launch_pack_attr(*g, c->attr, s);
  if (run_mlp) launches += launch_mlp_pack(*mlp, plan, c->mlp_blob, s);
  if (cudaMemsetAsync(c->control, 0, c->control_bytes, s) != cudaSuccess) return fail(c, SSSGS_ECUDA, "memset failed");
  uint32_t* cnt = c->gb.counters;
  launches += launch_project(*g, cam, c->gb, (flags & SSSGS_TIGHT_LISTS) ? 1 : 0, s);
  for (int p = 0; p < 4; ++p)
    launches += launch_depth_pass(c->gb.dkeys, c->gb.dvals, (uint32_t)n, p, c->gb.hist, c->status_depth[p],
                                  cnt + DC_TICKET_BASE + p, cnt + DC_SORT_ERROR, max_blocks, s);
  int tb = 1;
  while ((1 << tb) < tiles) ++tb;
  const int npass = tb > 8 ? 2 : 1;
  const int bits0 = npass == 2 ? (tb + 1) / 2 : tb, bits1 = npass == 2 ? tb - bits0 : 0;
  launches += launch_emit(n, cam, c->gb, cap, 0, bits0, bits0, bits1, c->status_emit, cnt + DC_TICKET_BASE + 4, s);
  launches += launch_sort_pass(c->gb.ikeys[0], c->gb.ivals[0], c->gb.ikeys[1], c->gb.ivals[1], cnt + DC_INSTANCES, cap, 0,
                               bits0, c->gb.hist + 4 * 256, c->status_tile[0], cnt + DC_TICKET_BASE + 5,
                               cnt + DC_SORT_ERROR, max_blocks, s);
  if (npass == 2)
    launches += launch_sort_pass(c->gb.ikeys[1], c->gb.ivals[1], c->gb.ikeys[0], c->gb.ivals[0], cnt + DC_INSTANCES, cap,
                                 bits0, bits1, c->gb.hist + 5 * 256, c->status_tile[1], cnt + DC_TICKET_BASE + 6,
                                 cnt + DC_SORT_ERROR, max_blocks, s);
  const int fi = npass & 1;
  const uint32_t* sorted_tiles = c->gb.ikeys[fi];
  const uint32_t* sorted_vals = c->gb.ivals[fi];
  launches += launch_ranges(sorted_tiles, cam, c->gb, cap, nullptr, gr->counters, 0, s);
  float* const input_grads[6] = {gr->grad_means, gr->grad_scales, gr->grad_rotations, gr->grad_attr,
                                 n_in == 2 ? gr->grad_feat : nullptr, n_in == 2 ? gr->grad_vis_sh : nullptr};
  // ---- per light batch -----------------------------------------------------------------------------
  for (int l0 = 0; l0 < n_light; l0 += c->max_lb) {
    const int nl = n_light - l0 < c->max_lb ? n_light - l0 : c->max_lb;
    LightBatch lb;
    memset(&lb, 0, sizeof lb);
    for (int l = 0; l < nl; ++l) {
      memcpy(lb.l[l].pos, lights[l0 + l].position, 12);
      memcpy(lb.l[l].intensity, lights[l0 + l].intensity, 12);
    }
    float4* mlp_buf = c->mlp_out[0];
    if (run_mlp) {
      const int k = launch_mlp(*g, plan, c->mlp_blob, cam, lb, nl, mlp_buf, nullptr, 0, c->num_sms, nullptr, nullptr, nullptr, s);
      if (k < 0) return fail(c, SSSGS_ECUDA, "MLP kernel configuration failed");
      launches += k;
    } else {
      launches += launch_gather_precomputed(mlp->precomputed_out + (int64_t)l0 * n * 4, n, nl, n * 4, mlp_buf, s);
    }
    launches += launch_shade_backward(cam, lb, nl, gr->gbuffer + (int64_t)l0 * npix * 16, gr->grad_rgb + (int64_t)l0 * npix * 3,
                                      gr->grad_gbuffer_in ? gr->grad_gbuffer_in + (int64_t)l0 * npix * 16 : nullptr,
                                      gr->grad_gbuffer + (int64_t)l0 * npix * 16, s);
    launches += launch_composite_backward(cam, nl, c->gb, sorted_vals, c->attr, mlp_buf, nl,
                                          gr->grad_gbuffer + (int64_t)l0 * npix * 16, gr->grad_opacity, gr->grad_mean2d,
                                          gr->grad_conic, gr->grad_depth, gr->grad_attr,
                                          gr->grad_mlp_out + (int64_t)l0 * n * 4, n, s);
    if (run_mlp && gr->grad_params)
      launches += launch_mlp_backward(*g, *mlp, cam, lb, nl, gr->grad_mlp_out + (int64_t)l0 * n * 4, gr->grad_params,
                                      reinterpret_cast<uint32_t*>(c->mlp_out[1]), cnt + DC_BWD_ROWS, c->bwd_blob,
                                      l0 == 0, (flags & SSSGS_BACKWARD_FP32) != 0, input_grads, c->num_sms, s);
  }
  // ---- a3 backward: the accumulated 2-D gradients through the projection ---------------------------
  if (n_geo == 3)
    launches += launch_project_backward(*g, cam, gr->grad_mean2d, gr->grad_conic, gr->grad_depth, gr->grad_means,
                                        gr->grad_scales, gr->grad_rotations, s);
  c->launches = launches;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, SSSGS_ECUDA, "CUDA error: %s", cudaGetErrorString(e));
  return SSSGS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Host-buffer entry point: one host->device crossing per call, results copied back.
// ---------------------------------------------------------------------------------------------
namespace {
void* stage_buf(sssgs_ctx* c, size_t idx, size_t bytes) {
  if (c->staging.size() <= idx) c->staging.resize(idx + 1, {nullptr, 0});
  auto& s = c->staging[idx];
  if (s.second < bytes || !s.first) {
    if (s.first) cudaFree(s.first);
    s.first = nullptr;
    s.second = 0;
    if (cudaMalloc(&s.first, bytes ? bytes : 16) != cudaSuccess) return nullptr;
    s.second = bytes ? bytes : 16;
  }
  return s.first;
}
}  // namespace

extern "C" int sssgs_render_host(sssgs_ctx* c, const sssgs_gaussians* g, const sssgs_mlp* mlp,
                                 const sssgs_camera* cams, int n_cam, const sssgs_light* lights,
                                 int n_light, const sssgs_out* out, uint32_t flags) {
  if (!c) return SSSGS_EINVAL;
  if (!g || !mlp || !out) return fail(c, SSSGS_EINVAL, "NULL argument");
  if (g->n < 0 || g->n > c->cfg.max_gaussians) return fail(c, SSSGS_ECAPACITY, "n out of range");
  if (n_cam < 0 || n_light < 0) return fail(c, SSSGS_EINVAL, "negative count");
  if (g->vis_sh_degree < 0 || g->vis_sh_degree > 1) return fail(c, SSSGS_EINVAL, "vis_sh_degree must be 0 or 1");
  if (g->feat_dim < 0 || g->feat_dim > 88 || g->feat_dim % 4) return fail(c, SSSGS_EINVAL, "feat_dim must be a multiple of 4 in [0,88]");
  // everything is validated BEFORE anything is staged or uploaded: a NULL host array must never be rendered
  // from uninitialised staging memory
  if ((n_cam > 0 && !cams) || (n_light > 0 && !lights)) return fail(c, SSSGS_EINVAL, "NULL argument");
  if (g->n > 0) {
    const void* req[] = {g->means, g->scales, g->rotations, g->opacities, g->normals, g->base_color,
                         g->roughness, g->metallic, g->subsurface, g->vis_sh};
    for (const void* p : req)
      if (!p) return fail(c, SSSGS_EINVAL, "a Gaussian attribute pointer is NULL");
    if (g->feat_dim > 0 && !g->feat) return fail(c, SSSGS_EINVAL, "feat is NULL");
  }
  if (!mlp->precomputed_out && g->n > 0 && n_light > 0 && n_cam > 0) {
    if (!mlp->params) return fail(c, SSSGS_EINVAL, "mlp.params is NULL");
    MlpPlan plan;  // checks the architecture and params_bytes against it
    const int rc = build_plan(c, *mlp, g->feat_dim, &plan);
    if (rc != SSSGS_OK) return rc;
  }
  for (int v = 1; v < n_cam; ++v)
    if (cams[v].width != cams[0].width || cams[v].height != cams[0].height)
      return fail(c, SSSGS_EINVAL, "sssgs_render_host: all cameras of a call must share one image size");
  DeviceGuard guard(c->cfg.device);
  if (!guard.ok) return fail(c, SSSGS_ECUDA, "cudaSetDevice(%d) failed", c->cfg.device);
  cudaStream_t s = 0;
  const size_t n = (size_t)g->n;
  const size_t ncoef = (size_t)(g->vis_sh_degree + 1) * (g->vis_sh_degree + 1);
  size_t idx = 0;
  bool ok = true;
  // What projection / sort / binning read goes up first, on the stream the render runs on; the
  // rest (what only the MLP and the attribute packing read) goes up on the context's copy stream,
  // so that the geometry chain runs under the second part of the upload.
  cudaStream_t up_stream = s;
  auto up = [&](const void* host, size_t bytes) -> void* {
    void* d = stage_buf(c, idx++, bytes);
    if (!d) { ok = false; return nullptr; }
    if (host && bytes && cudaMemcpyAsync(d, host, bytes, cudaMemcpyHostToDevice, up_stream) != cudaSuccess) ok = false;
    return d;
  };
  sssgs_gaussians dg = *g;
  dg.means = (const float*)up(g->means, n * 12);
  dg.scales = (const float*)up(g->scales, n * 12);
  dg.rotations = (const float*)up(g->rotations, n * 16);
  dg.opacities = (const float*)up(g->opacities, n * 4);
  const bool split = mlp->precomputed_out == nullptr && n > 0 && n_light > 0 && n_cam > 0;
  if (split) up_stream = c->copy;
  dg.normals = (const float*)up(g->normals, n * 12);
  dg.base_color = (const float*)up(g->base_color, n * 12);
  dg.roughness = (const float*)up(g->roughness, n * 4);
  dg.metallic = (const float*)up(g->metallic, n * 4);
  dg.subsurface = (const float*)up(g->subsurface, n * 4);
  dg.vis_sh = (const float*)up(g->vis_sh, n * ncoef * 4);
  dg.feat = (const float*)up(g->feat_dim ? g->feat : nullptr, n * (size_t)g->feat_dim * 4);
  sssgs_mlp dm = *mlp;
  dm.params = up(mlp->params, mlp->params ? mlp->params_bytes : 0);
  const size_t frames = (size_t)n_cam * n_light;
  dm.precomputed_out = mlp->precomputed_out ? (const float*)up(mlp->precomputed_out, frames * n * 16) : nullptr;
  if (!mlp->precomputed_out) idx++;
  if (split) {
    if (cudaEventRecord(c->ev_upload, c->copy) != cudaSuccess) ok = false;
    c->upload_pending = true;
  }

  size_t npix = 0, tiles = 0;  // all cameras of one call share the frame size of the first
  if (n_cam > 0 && cams) {
    npix = (size_t)cams[0].width * cams[0].height;
    tiles = (size_t)((cams[0].width + kTile - 1) / kTile) * ((cams[0].height + kTile - 1) / kTile);
  }
  const size_t cap = (size_t)c->cfg.max_instances;
  struct Back { void* host; void* dev; size_t bytes; };
  std::vector<Back> back;
  auto down = [&](void* host, size_t bytes) -> void* {
    if (!host) { idx++; return nullptr; }
    void* d = stage_buf(c, idx++, bytes);
    if (!d) { ok = false; return nullptr; }
    back.push_back({host, d, bytes});
    return d;
  };
  sssgs_out dout;
  dout.rgb = (float*)down(out->rgb, ((flags & SSSGS_SUM_LIGHTS) ? (size_t)n_cam : frames) * npix * 12);
  dout.gbuffer = (float*)down(out->gbuffer, frames * npix * 64);
  dout.aov_diffuse = (float*)down(out->aov_diffuse, frames * npix * 12);
  dout.aov_specular = (float*)down(out->aov_specular, frames * npix * 12);
  dout.mlp_out = (float*)down(out->mlp_out, frames * n * 16);
  dout.sorted_keys = (uint64_t*)down(out->sorted_keys, (size_t)n_cam * cap * 8);
  dout.sorted_vals = (uint32_t*)down(out->sorted_vals, (size_t)n_cam * cap * 4);
  dout.tile_ranges = (uint32_t*)down(out->tile_ranges, (size_t)n_cam * tiles * 8);
  // counters are always fetched: they carry the overflow flag
  std::vector<int64_t> cnt_host((size_t)(n_cam > 0 ? n_cam : 1) * SSSGS_NCOUNTERS, 0);
  dout.counters = (int64_t*)stage_buf(c, idx++, cnt_host.size() * 8);
  if (!dout.counters) ok = false;
  // error paths after the uploads were enqueued: the copies read caller memory, so they are drained and the
  // pending-upload mark is cleared before returning
  auto drain = [&]() {
    cudaStreamSynchronize(c->copy);
    cudaStreamSynchronize(s);
    c->upload_pending = false;
  };
  if (!ok) {
    const cudaError_t e = cudaGetLastError();
    drain();
    return fail(c, SSSGS_ECUDA, "device staging allocation or upload failed: %s", cudaGetErrorString(e));
  }

  const int rc = sssgs_render(c, &dg, &dm, cams, n_cam, lights, n_light, &dout, flags, s);
  if (rc != SSSGS_OK) {
    const std::string msg = c->err;
    drain();
    c->err = msg;
    return rc;
  }
  for (const Back& b : back)
    if (b.bytes && cudaMemcpyAsync(b.host, b.dev, b.bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess)
      return fail(c, SSSGS_ECUDA, "download failed");
  if (n_cam > 0 && cudaMemcpyAsync(cnt_host.data(), dout.counters, (size_t)n_cam * SSSGS_NCOUNTERS * 8, cudaMemcpyDeviceToHost, s) != cudaSuccess)
    return fail(c, SSSGS_ECUDA, "download failed");
  const cudaError_t e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(c, SSSGS_ECUDA, "CUDA error: %s", cudaGetErrorString(e));
  for (int v = 0; v < n_cam; ++v) {
    if (out->counters) memcpy(out->counters + (size_t)v * SSSGS_NCOUNTERS, cnt_host.data() + (size_t)v * SSSGS_NCOUNTERS, SSSGS_NCOUNTERS * 8);
    if (cnt_host[(size_t)v * SSSGS_NCOUNTERS + SSSGS_CNT_SORT_ERROR]) return fail(c, SSSGS_ECUDA, "internal: look-back wait exceeded its bound (camera %d)", v);
    if (cnt_host[(size_t)v * SSSGS_NCOUNTERS + SSSGS_CNT_OVERFLOW])
      return fail(c, SSSGS_EOVERFLOW, "camera %d: %lld tile instances exceed max_instances %lld", v,
                  (long long)cnt_host[(size_t)v * SSSGS_NCOUNTERS + SSSGS_CNT_INSTANCES], (long long)cap);
  }
  return SSSGS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// sssgs_mlp_eval_static: the per-Gaussian MLP (steps a1 + a2) without a context and without any allocation.
//
// The tensor-core MLP kernel does not read the caller's fp32 parameters: mlp_pack_kernel first rewrites them as
// swizzled 16-bit UMMA operands (weights + split biases) into a global-memory scratch block, and every CTA of
// mlp_kernel pulls that block into shared memory.  In the render path the block lives in the context's
// workspace (cudaMalloc'ed by sssgs_create unless the caller brings one).  Here it lives in the array below,
// which is part of the library's device image: the driver places it when the module is loaded on a device and
// it stays there until the process exits.
//
// g_static_blob is only a handle on the host side.  Host code that hands `g_static_blob` itself to a kernel
// passes the address of a host shadow object, not device memory: the kernel would fault (or, on machines where
// the GPU can dereference host addresses, quietly work on the wrong bytes).  The device address has to be asked
// for, per device, with that device current: cudaGetSymbolAddress.  static_scratch_for() does that once per
// device ordinal and remembers the answer.
// ---------------------------------------------------------------------------------------------------------
namespace {

static __device__ __align__(256) uint8_t g_static_blob[SSSGS_STATIC_SCRATCH_BYTES];

constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
  bool ready = false;
  uint8_t* blob = nullptr;  // device address of g_static_blob on this device
  int num_sms = 0;
};
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

// Must be called with `device` current.  First call per device: resolves the array's device address and reads
// the SM count; later calls only read the cached values.
int static_scratch_for(int device, StaticDevice* out) {
  if (device < 0 || device >= kStaticMaxDevices)
    return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: device ordinal %d outside [0, %d)", device, kStaticMaxDevices);
  std::lock_guard<std::mutex> lock(g_static_mu);
  StaticDevice& d = g_static_dev[device];
  if (!d.ready) {
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess)
      return fail(nullptr, SSSGS_ECUDA, "sssgs_mlp_eval_static: cannot query device %d (libsssgs has no CPU fallback)", device);
    if (major != 10)
      return fail(nullptr, SSSGS_EARCH, "sssgs_mlp_eval_static: device %d is sm_%dx; libsssgs is built for sm_100a only", device, major);
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_blob);
    if (e != cudaSuccess || !p)
      return fail(nullptr, SSSGS_ECUDA, "sssgs_mlp_eval_static: cudaGetSymbolAddress failed on device %d: %s", device,
                  cudaGetErrorString(e));
    d.blob = static_cast<uint8_t*>(p);
    d.num_sms = sms;
    d.ready = true;
  }
  *out = d;
  return SSSGS_OK;
}

}  // namespace

extern "C" int sssgs_mlp_eval_static(int device, const sssgs_gaussians* g, const sssgs_mlp* mlp,
                                     const sssgs_camera* cam, const sssgs_light* lights, int n_light,
                                     float* mlp_out, void* cuda_stream) {
  if (!g || !mlp || !cam || (n_light > 0 && !lights)) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: NULL argument");
  if (n_light < 0) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: negative light count");
  if (n_light > SSSGS_STATIC_MAX_LIGHTS)
    return fail(nullptr, SSSGS_ECAPACITY, "sssgs_mlp_eval_static: n_light %d > SSSGS_STATIC_MAX_LIGHTS (%d); call once per batch of lights",
                n_light, SSSGS_STATIC_MAX_LIGHTS);
  if (g->n < 0) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: n < 0");
  if (g->n > (int64_t)1 << 30) return fail(nullptr, SSSGS_ECAPACITY, "sssgs_mlp_eval_static: n %lld > 2^30", (long long)g->n);
  if (g->vis_sh_degree < 0 || g->vis_sh_degree > 1) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: vis_sh_degree must be 0 or 1");
  if (g->feat_dim < 0 || g->feat_dim > 88 || g->feat_dim % 4)
    return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: feat_dim must be a multiple of 4 in [0,88]");
  if (g->n > 0) {
    // the arrays the MLP's input row is assembled from (Eq. 6); the others are not read
    const void* req[] = {g->means, g->scales, g->rotations, g->normals, g->vis_sh};
    for (const void* p : req)
      if (!p || !aligned16(p))
        return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: means / scales / rotations / normals / vis_sh is NULL or not 16-byte aligned");
    if (g->feat_dim > 0 && (!g->feat || !aligned16(g->feat))) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: feat is NULL or misaligned");
    if (n_light > 0 && (!mlp_out || !aligned16(mlp_out))) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: mlp_out is NULL or misaligned");
  }
  if (mlp->precomputed_out) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: mlp.precomputed_out must be NULL");
  if (!mlp->params || !aligned16(mlp->params)) return fail(nullptr, SSSGS_EINVAL, "sssgs_mlp_eval_static: mlp.params is NULL or misaligned");
  MlpPlan plan;
  const int rc = build_plan(nullptr, *mlp, g->feat_dim, &plan);
  if (rc != SSSGS_OK) return rc;
  if ((size_t)plan.blob_bytes > (size_t)SSSGS_STATIC_SCRATCH_BYTES)
    return fail(nullptr, SSSGS_ECAPACITY,
                "sssgs_mlp_eval_static: the packed weights of this MLP take %d bytes, the static scratch holds %d "
                "(SSSGS_STATIC_SCRATCH_BYTES); use sssgs_render with a context for larger networks",
                plan.blob_bytes, (int)SSSGS_STATIC_SCRATCH_BYTES);
  if (g->n == 0 || n_light == 0) return SSSGS_OK;

  DeviceGuard guard(device);
  if (!guard.ok) return fail(nullptr, SSSGS_ECUDA, "sssgs_mlp_eval_static: cudaSetDevice(%d) failed", device);
  StaticDevice dev;
  const int rs = static_scratch_for(device, &dev);
  if (rs != SSSGS_OK) return rs;

  cudaStream_t s = (cudaStream_t)cuda_stream;
  const CamParams cp = make_cam(*cam);  // only the camera position (w_out) enters the MLP
  LightBatch lb;
  memset(&lb, 0, sizeof lb);
  for (int l = 0; l < n_light; ++l) {
    memcpy(lb.l[l].pos, lights[l].position, 12);
    memcpy(lb.l[l].intensity, lights[l].intensity, 12);
  }
  // Nothing in the block has to start at zero: the pack kernel rewrites every byte of the operand and bias
  // tiles of THIS plan (zero padding included), and the bytes between / behind them, which may still hold the
  // previous call's network, are copied to shared memory but never addressed by an MMA descriptor.
  launch_mlp_pack(*mlp, plan, dev.blob, s);
  const int k = launch_mlp(*g, plan, dev.blob, cp, lb, n_light, reinterpret_cast<float4*>(mlp_out), nullptr, 0,
                           dev.num_sms, nullptr, nullptr, nullptr, s);
  if (k < 0) return fail(nullptr, SSSGS_ECUDA, "sssgs_mlp_eval_static: MLP kernel configuration failed: %s", cudaGetErrorString(cudaGetLastError()));
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, SSSGS_ECUDA, "sssgs_mlp_eval_static: CUDA error: %s", cudaGetErrorString(e));
  return SSSGS_OK;
}

// SURVEY 8(f).1, second half: relighting from a precomputed reflectance field.  Needs no context
// and no scratch: a streaming sum over the OLAT stack.
extern "C" int sssgs_relight(int device, const float* frames, int n_light, int64_t n_pixels, const float* weights,
                             float* out, void* cuda_stream) {
  if (n_light < 0 || n_pixels < 0) return fail(nullptr, SSSGS_EINVAL, "sssgs_relight: negative count");
  if (n_pixels > ((int64_t)1 << 40) / 12) return fail(nullptr, SSSGS_ECAPACITY, "sssgs_relight: n_pixels too large");
  if (n_pixels == 0) return SSSGS_OK;
  if (!out || !aligned16(out)) return fail(nullptr, SSSGS_EINVAL, "sssgs_relight: out is NULL or not 16-byte aligned");
  if (n_light > 0 && (!frames || !weights || !aligned16(frames)))
    return fail(nullptr, SSSGS_EINVAL, "sssgs_relight: frames / weights NULL or frames not 16-byte aligned");
  if (n_light > 0) {   // out must not overlap the stack it is computed from
    const char* f0 = (const char*)frames;
    const char* f1 = f0 + (size_t)n_light * n_pixels * 12;
    const char* o0 = (const char*)out;
    if (o0 < f1 && o0 + (size_t)n_pixels * 12 > f0) return fail(nullptr, SSSGS_EINVAL, "sssgs_relight: out overlaps frames");
  }
  DeviceGuard guard(device);
  if (!guard.ok) return fail(nullptr, SSSGS_ECUDA, "sssgs_relight: cudaSetDevice(%d) failed", device);
  int major = 0, sms = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess)
    return fail(nullptr, SSSGS_ECUDA, "sssgs_relight: cannot query device %d (libsssgs has no CPU fallback)", device);
  if (major != 10) return fail(nullptr, SSSGS_EARCH, "sssgs_relight: device %d is sm_%dx; libsssgs is built for sm_100a only", device, major);
  launch_relight(frames, n_light, n_pixels, weights, out, sms, (cudaStream_t)cuda_stream);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, SSSGS_ECUDA, "sssgs_relight: CUDA error: %s", cudaGetErrorString(e));
  return SSSGS_OK;
}
