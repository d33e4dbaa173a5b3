// C-ABI entry points of libspense (include/spense.h): argument checking, stream-K schedule,
// tensor-map creation and launches.  No device allocation, no synchronisation and no device reads in the GEMM calls.
#include <cudaTypedefs.h>

#include <cstdlib>
#include <cstring>
#include <deque>
#include <mutex>
#include <vector>

#include "spense_internal.cuh"

namespace spense {
namespace {

// ---- per-process / per-device state.  One entry per device ordinal; nothing assumes a single device.
struct Device { int probed = 0, arch_ok = 0, sms = 0; };
std::mutex g_dev_mu;
Device g_dev[64];
PFN_cuTensorMapEncodeTiled_v12000 g_encode = nullptr;
int* g_status = nullptr;        // mapped pinned host word: the first device-side error (see spense_device_status)
#ifdef SPENSE_DEBUG_HOOKS
long long* g_trace = nullptr;   // debug: set by spense_debug_set_trace
#endif

int check_device(int* dev_out, int* sms_out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return SPENSE_ERR_CUDA;
  std::lock_guard<std::mutex> lk(g_dev_mu);
  Device& d = g_dev[dev];
  if (!d.probed) {
    int major = 0, minor = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
    cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
    if (d.sms > kMaxSpans) d.sms = kMaxSpans;   // the persistent CTAs of a launch own fix-up slots 0..kMaxSpans-1
    d.arch_ok = (major == 10 && minor == 0) ? 1 : 0;
    d.probed = 1;
  }
  if (!d.arch_ok) return SPENSE_ERR_ARCH;
  if (!g_encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return SPENSE_ERR_CUDA;
    g_encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  }
  if (!g_status) {
    void* h = nullptr;
    if (cudaHostAlloc(&h, 64, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) return SPENSE_ERR_CUDA;
    std::memset(h, 0, 64);
    g_status = reinterpret_cast<int*>(h);
  }
  if (dev_out) *dev_out = dev;
  if (sms_out) *sms_out = d.sms;
  return SPENSE_OK;
}

// a device-side error recorded by an earlier launch (bad blob header, a CTA that gave up waiting for its peers)
int pending_device_error() {
  return g_status ? *reinterpret_cast<volatile int*>(g_status) : SPENSE_OK;
}

int check_shape(const spense_shape_t* s) {
  if (!s) return SPENSE_ERR_ARG;
  if (s->H < 128 || s->I < 128 || s->I_dense < 0 || s->I_dense > s->I) return SPENSE_ERR_SHAPE;
  if (s->H % 128 || s->I % 128 || s->I_dense % 128) return SPENSE_ERR_SHAPE;
  if (s->H > (1 << 20) || s->I > (1 << 20)) return SPENSE_ERR_SHAPE;
  return SPENSE_OK;
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// tuning knobs exist in SPENSE_DEBUG_HOOKS builds only (experiments); the shipped library reads no environment variable
#ifdef SPENSE_DEBUG_HOOKS
int knob(const char* name, int dflt) { const char* e = std::getenv(name); return e ? std::atoi(e) : dflt; }
#else
constexpr int knob(const char*, int dflt) { return dflt; }
#endif

// ---- launch geometry.  Every call runs on CTA pairs (spense_gemm.cu): token blocks of at most kWideMaxTokens tokens (one
// block of kWideMaxTokens1 for 241..256 tokens), `par` blocks side by side in one launch with pairs / par stream-K spans
// each (the pairs of different blocks walk the same schedule, so a weight stage is read from HBM once and found in L2 by
// the other blocks); more blocks than fit run as further launches.
struct Plan {
  int n_pad;      // token columns of one block
  int nb;         // token blocks
  int par;        // blocks per launch
  int spans;      // stream-K spans per block (CTA pairs)
  int ring;       // stage-ring slots
  int slot_bytes;
};

int ring_of(int n_pad, int* slot_bytes) {
  const int slot = kSparseOperandBytes + (n_pad / 2) * 256;          // one operand (values + metadata) + two half token tiles
  const int stages = (kSmemMax - 1024 - 256 - 20 * n_pad) / slot;   // barriers + the scale tables
  if (slot_bytes) *slot_bytes = slot;
  return stages > 8 ? 8 : stages;
}

// how many of `nb` blocks one launch takes.  In units of the time one token block needs on all `units` CTA pairs, a launch
// of c blocks with k = units / c spans each costs c * units / (c * k) (some pairs idle when c does not divide units) plus
// about one unit of its own: every launch re-streams the weights from HBM, ramps up and ends with a fix-up tail.  The
// split with the smallest total wins, the larger c on a tie.  (An earlier rule -- the largest c within 5 % of the best
// occupancy -- picked c = 2 for 35 blocks because c = 1 wastes nothing: M = 8192 ran as 18 launches.)
int par_of(int nb, int units, int cap) {
  auto cost = [&](int c) {
    const int rounds = (nb + c - 1) / c, k = units / c;
    return rounds * ((double)c * units / (c * k) + 1.0);
  };
  int cmax = nb < units ? nb : units;
  if (cmax > cap) cmax = cap;
  int pick = 1;
  for (int c = 2; c <= cmax; ++c)
    if (cost(c) <= cost(pick) + 1e-9) pick = c;
  return pick;
}

// act_row_bytes: bytes of one token row of the activation operand (H for gate_up, I for down).  The token tiles of the
// blocks of one launch are re-read from L2 once per weight tile, so a launch takes only as many blocks as keep that
// working set (blocks x n_pad x act_row_bytes) well inside the 126 MB L2: measured at M = 8192, 18 blocks of Hq (110 MB)
// side by side made down HBM-bound on activation re-reads (1020 us against 4 x 167 us at M = 2048).
constexpr size_t kActWorkingSetBytes = 64u << 20;
Plan plan_of(int M, int sms, int act_row_bytes, bool in_split) {
  Plan pl = {};
  pl.nb = M <= kWideMaxTokens1 ? 1 : (M + kWideMaxTokens - 1) / kWideMaxTokens;
  // input-split walks (down): two blocks side by side leave 37 spans over the row tiles, every tile then splits three ways
  // and ends in the reduce-scatter with large partials; three blocks (24 spans) split two ways, which the TMEM preload
  // handles (measured: M = 300 down 67 -> 59 us, M = 480 82 -> 66 us; gate_up prefers the larger blocks: 62.6 vs 81.3 us)
  if (in_split && pl.nb == 2) pl.nb = 3;
  pl.n_pad = ((M + pl.nb - 1) / pl.nb + 15) / 16 * 16;
  const int pairs = sms / 2;
  size_t cap = ((size_t)knob("SPENSE_ACT_WS_MB", (int)(kActWorkingSetBytes >> 20)) << 20) / ((size_t)pl.n_pad * act_row_bytes);
  cap = cap < 1 ? 1 : (cap > 12 ? 12 : cap);
  pl.par = par_of(pl.nb, pairs, (int)cap);
  pl.spans = pairs / pl.par;
  pl.ring = ring_of(pl.n_pad, &pl.slot_bytes);
  return pl;
}

// token columns whose partials the workspace must hold at up to M tokens (monotone in M: 241..256 tokens run as one block)
size_t ws_bytes_for(int M) {
  const size_t cols = M >= kWideMaxTokens1 ? (size_t)kWideMaxTokens1 : (size_t)((M + 15) / 16 * 16);
  return kWsFixedBytes + (size_t)kMaxSpans * 2 * cols * 128 * sizeof(float);
}

// ---- stream-K schedule: cut the stage sequence into n_spans spans of (nearly) equal cost.
struct Schedule {
  int mode, H, I, I_d, n_pad, spans_req, ring, nb;
  int n_spans;
  int span_begin[kMaxSpans + 1];
  uint32_t span_off[kMaxSpans];   // byte offset of the span's first stage image inside its section
  uint32_t span_pre[kMaxSpans];   // bytes of the stages the producer issues before anything else (one ring)
  uint32_t span_len[kMaxSpans];   // bytes of the whole span
};

std::mutex g_sched_mu;
std::deque<Schedule> g_sched;   // deque: references handed out stay valid

const Schedule& get_schedule(int mode, const Geometry& g, const Plan& pl) {
  std::lock_guard<std::mutex> lk(g_sched_mu);
  for (const Schedule& s : g_sched)
    if (s.mode == mode && s.H == g.H && s.I == g.I && s.I_d == g.I_d && s.n_pad == pl.n_pad && s.spans_req == pl.spans &&
        s.ring == pl.ring && s.nb == pl.nb)
      return s;
  Schedule sc = {};
  sc.mode = mode; sc.H = g.H; sc.I = g.I; sc.I_d = g.I_d; sc.n_pad = pl.n_pad; sc.spans_req = pl.spans; sc.ring = pl.ring; sc.nb = pl.nb;
  // cost of a stage.  Every CTA keeps the same number of ring slots in flight, so under HBM contention a
  // stage costs one slot latency plus its bytes: measured on B200 (profiles/) a 40 KB sparse stage takes
  // ~1.12x a 32 KB dense one => fixed part ~36 KB-equivalents; activation bytes come from L2 and weigh less.
  // From three token blocks on (M > 480) a launch is paced by the tensor pipe instead: a sparse stage (K 256) and a
  // dense one (K 128) issue the same four MMAs.
  const double fixed = knob("SPENSE_SCHED_FIXED", 36864), gamma = knob("SPENSE_SCHED_GAMMA_PCT", 25) / 100.0;
  const bool tensor_paced = pl.nb > 2;
  const double cs = tensor_paced ? 1.0 : fixed + kSparseStageBytes + gamma * 2.0 * pl.n_pad * 128;
  const double cd = tensor_paced ? 1.0 : fixed + kDenseStageBytes + gamma * 1.0 * pl.n_pad * 128;
  std::vector<double> cost;
  if (mode != 1) {
    cost.insert(cost.end(), (size_t)g.gu_tiles_sparse * g.gu_ns, cs);
    cost.insert(cost.end(), (size_t)(g.gu_tiles - g.gu_tiles_sparse) * g.gu_nd, cd);
  } else {
    for (int t = 0; t < g.dn_tiles; ++t) {
      cost.insert(cost.end(), (size_t)g.dn_ns, cs);
      cost.insert(cost.end(), (size_t)g.dn_nd, cd);
    }
  }
  const int total = (int)cost.size();
  int spans = pl.spans < kMaxSpans ? pl.spans : kMaxSpans;
  if (spans > total) spans = total;
  double sum = 0;
  for (double c : cost) sum += c;
  sc.n_spans = spans;
  double acc = 0;
  int s = 0;
  sc.span_begin[0] = 0;
  for (int i = 1; i < spans; ++i) {
    const double target = sum * (double)i / spans;
    while (s < total && acc + 0.5 * cost[s] < target) acc += cost[s++];
    int b = s;
    if (b <= sc.span_begin[i - 1]) b = sc.span_begin[i - 1] + 1;     // every span owns >= 1 stage
    if (b > total - (spans - i)) b = total - (spans - i);
    while (s < b) acc += cost[s++];
    sc.span_begin[i] = b;
  }
  sc.span_begin[spans] = total;
  // byte offsets: the blob stores the stage images in exactly this linear order
  std::vector<uint32_t> bytes(total);
  if (mode != 1) {
    for (int i = 0; i < total; ++i) bytes[i] = i < g.gu_tiles_sparse * g.gu_ns ? kSparseStageBytes : kDenseStageBytes;
  } else {
    const int per = g.dn_ns + g.dn_nd;
    for (int i = 0; i < total; ++i) bytes[i] = (i % per) < g.dn_ns ? kSparseStageBytes : kDenseStageBytes;
  }
  uint64_t off = 0;
  int st = 0;
  for (int i = 0; i < spans; ++i) {
    while (st < sc.span_begin[i]) off += bytes[st++];
    sc.span_off[i] = (uint32_t)off;
    uint32_t pre = 0;
    for (int k = sc.span_begin[i]; k < sc.span_begin[i + 1] && k < sc.span_begin[i] + pl.ring; ++k) pre += bytes[k];
    sc.span_pre[i] = pre;
    uint32_t len = 0;
    for (int k = sc.span_begin[i]; k < sc.span_begin[i + 1]; ++k) len += bytes[k];
    sc.span_len[i] = len;
  }
  g_sched.push_back(sc);
  return g_sched.back();
}

// uint8 tensor [rows, K] row-major; box = 128 bytes of K x box_rows rows, 128-byte swizzle (activation tiles)
int make_tmap(CUtensorMap* map, const uint8_t* base, int K, int rows, int box_rows) {
  cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)K};
  cuuint32_t box[2] = {128u, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = g_encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? SPENSE_OK : SPENSE_ERR_CUDA;
}

// a blob section seen as rows of 128 bytes; box = one operand of a stage image (already swizzled: plain copy).  Lets a
// CTA of a pair fetch its operand with a tensor copy whose completion counts on the LEADER CTA's barrier.
int make_tmap_section(CUtensorMap* map, const uint8_t* base, size_t bytes, int box_rows) {
  cuuint64_t dims[2] = {128u, (cuuint64_t)(bytes / 128)};
  cuuint64_t strides[1] = {128u};
  cuuint32_t box[2] = {128u, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = g_encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? SPENSE_OK : SPENSE_ERR_CUDA;
}

// bytes of span k that the PREVIOUS launch pulls into L2 during its tail: at least one ring
constexpr uint32_t kPfNextBytes = 1280u * 1024u;   // B200 sweep (M = 64, us/layer): 160 KB 54.2, 640 KB 53.6, 1280 KB 52.6, 2560 KB 53.0
constexpr int kPfPaceNs = 1500;                    // per 32 KB chunk and CTA; 300 ns: 56.0, 750: 52.7, 1500: 52.5
uint32_t next_prefetch_bytes(const Schedule& sc, int k) {
  const uint32_t want = (uint32_t)knob("SPENSE_PF_NEXT_KB", kPfNextBytes / 1024) * 1024u;
  uint32_t n = sc.span_pre[k] > want ? sc.span_pre[k] : want;
  return n < sc.span_len[k] ? n : sc.span_len[k];
}

void fill_common(GemmParams& p, const Schedule& sc, const Plan& pl, const spense_shape_t* shape, const void* d_blob, int M, void* d_ws) {
#ifdef SPENSE_DEBUG_HOOKS
  p.trace = g_trace;
  if (g_trace) g_trace += (size_t)kMaxSpans * 16;   // debug: consecutive launches fill consecutive timelines
  { const char* e = std::getenv("SPENSE_DBG"); p.dbg = e ? std::atoi(e) : 0; }
#endif
  p.hdr = reinterpret_cast<const BlobHeader*>(d_blob);
  p.H = shape->H; p.I = shape->I; p.I_d = shape->I_dense;
  p.status = g_status;
  p.n_spans = sc.n_spans;
  std::memcpy(p.span_begin, sc.span_begin, sizeof(int) * (sc.n_spans + 1));
  p.nb = 1;
  p.blk0 = 0;
  p.M = M;
  p.n_pad = pl.n_pad;
  p.slot_bytes = pl.slot_bytes;
  p.num_stages = pl.ring;
  p.acc_stride = pl.n_pad > kWideMaxTokens ? kWideMaxTokens1 : kWideMaxTokens;   // 2 buffers x 240 columns (or 1 x 256), metadata at 480
  p.num_acc_bufs = pl.n_pad > kWideMaxTokens ? 1 : 2;
  uint8_t* ws = reinterpret_cast<uint8_t*>(d_ws);
  p.ws_ctrl = reinterpret_cast<int*>(ws);
  p.flags = reinterpret_cast<int*>(ws + 128);
  p.partials = reinterpret_cast<float*>(ws + kWsFixedBytes);
}

// L2 prefetch hint: while this launch runs its fix-up tail, pull what the next launch streams first.
void fill_next(GemmParams& p, const uint8_t* next_section, const Schedule& next) {
  if (!next_section) return;
  p.next_base = next_section;
  p.pf_pace_ns = knob("SPENSE_PF_PACE_NS", kPfPaceNs);
  for (int i = 0; i < p.n_spans; ++i) {
    const int k = i < next.n_spans ? i : next.n_spans - 1;
    p.next_off[i] = next.span_off[k];
    p.next_len[i] = i < next.n_spans ? next_prefetch_bytes(next, k) : 0;
  }
}

struct Launch { int dev, sms; };

// gate_up over all M tokens (one or several launches); dynamic: h stays in fp32, max|h| per slot goes to the workspace
int gate_up_impl(const Launch& L, const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t M,
                 const float* d_sh, int32_t sh_stride, uint8_t* d_hq, float* d_h_f32, void* d_ws, bool pdl, bool down_follows,
                 cudaStream_t stream, bool dynamic = false, float* d_sh_out = nullptr) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const Plan pl = plan_of(M, L.sms, g.H, false);
  const Schedule& sc = get_schedule(0, g, pl);
  const uint8_t* section = reinterpret_cast<const uint8_t*>(d_blob) + g.gate_up_off;
  CUtensorMap tm, tws, twd;
  int st = make_tmap(&tm, d_x, g.H, M, pl.n_pad / 2);
  if (!st) st = make_tmap_section(&tws, section, g.down_off - g.gate_up_off, kSparseOperandBytes / 128);
  if (!st) st = make_tmap_section(&twd, section, g.down_off - g.gate_up_off, kOperandBytes / 128);
  if (st) return st;
  for (int blk0 = 0; blk0 < pl.nb; blk0 += pl.par) {
    GemmParams p = {};
    fill_common(p, sc, pl, shape, d_blob, M, d_ws);
    p.nb = pl.nb - blk0 < pl.par ? pl.nb - blk0 : pl.par;
    p.blk0 = blk0;
    p.section = section;
    p.mode = 0;
    p.num_tiles = g.gu_tiles; p.tiles_sparse = g.gu_tiles_sparse;
    p.ns = g.gu_ns; p.nd = g.gu_nd; p.dense_k0 = 0;
    p.s_act = d_sx;
    p.s_h = d_sh; p.sh_stride = sh_stride;
    p.scale0 = 0; p.scale1 = 1;
    p.hq = d_hq;
    p.h_f32 = d_h_f32;
    p.amax_part = dynamic ? reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(d_ws) + kFlagBytes) : nullptr;
    p.ld_out = g.I; p.out_rows = g.I;
    if (down_follows && blk0 + pl.par >= pl.nb)                // the same layer's down projection streams next
      fill_next(p, reinterpret_cast<const uint8_t*>(d_blob) + g.down_off, get_schedule(1, g, plan_of(M, L.sms, g.I, true)));
    st = launch_gemm(p, tm, tws, twd, pdl, L.dev, stream);
    if (st) return st;
    if (dynamic) {
      // rows of this launch: s_h = max over the block's slots / 448, Hq = E4M3(h / s_h)
      const int m0 = blk0 * pl.n_pad;
      const int rows = (M - m0) < p.nb * pl.n_pad ? (M - m0) : p.nb * pl.n_pad;
      const int slots_per_block = 2 * sc.n_spans;
      st = launch_requant_rows(d_h_f32 + (size_t)m0 * g.I, rows, g.I, p.amax_part, slots_per_block, pl.n_pad, pl.n_pad,
                               d_hq + (size_t)m0 * g.I, d_sh_out + m0, L.sms, stream);
      if (st) return st;
    }
  }
  return SPENSE_OK;
}

int down_impl(const Launch& L, const spense_shape_t* shape, const void* d_blob, const uint8_t* d_hq, const float* d_sh,
              int32_t sh_stride, int32_t M, void* d_y, int32_t y_dtype, void* d_ws, bool pdl, const void* d_next_blob,
              cudaStream_t stream) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const Plan pl = plan_of(M, L.sms, g.I, true);
  const Schedule& sc = get_schedule(1, g, pl);
  const uint8_t* section = reinterpret_cast<const uint8_t*>(d_blob) + g.down_off;
  CUtensorMap tm, tws, twd;
  int st = make_tmap(&tm, d_hq, g.I, M, pl.n_pad / 2);
  if (!st) st = make_tmap_section(&tws, section, g.total_bytes - g.down_off, kSparseOperandBytes / 128);
  if (!st) st = make_tmap_section(&twd, section, g.total_bytes - g.down_off, kOperandBytes / 128);
  if (st) return st;
  for (int blk0 = 0; blk0 < pl.nb; blk0 += pl.par) {
    GemmParams p = {};
    fill_common(p, sc, pl, shape, d_blob, M, d_ws);
    p.nb = pl.nb - blk0 < pl.par ? pl.nb - blk0 : pl.par;
    p.blk0 = blk0;
    p.section = section;
    p.mode = 1;
    p.num_tiles = g.dn_tiles; p.tiles_sparse = 0;
    p.ns = g.dn_ns; p.nd = g.dn_nd; p.dense_k0 = g.I_s;
    p.s_act = d_sh; p.sh_stride = sh_stride;
    p.scale0 = 2; p.scale1 = 2;
    p.y = d_y;
    p.y_dtype = y_dtype;
    p.ld_out = g.H; p.out_rows = g.H;
    if (d_next_blob && blk0 + pl.par >= pl.nb)                 // the next layer's gate/up weights stream next
      fill_next(p, reinterpret_cast<const uint8_t*>(d_next_blob) + g.gate_up_off, get_schedule(0, g, plan_of(M, L.sms, g.H, false)));
    st = launch_gemm(p, tm, tws, twd, pdl, L.dev, stream);
    if (st) return st;
  }
  return SPENSE_OK;
}

// ---- stand-alone linears (spense_pack_linear blobs): in-split = the down walk, out-split = the gate_up walk with the plain epilogue
int check_linear_shape(const spense_linear_shape_t* s) {
  if (!s) return SPENSE_ERR_ARG;
  if (s->split != SPENSE_SPLIT_OUT && s->split != SPENSE_SPLIT_IN) return SPENSE_ERR_ARG;
  if (s->N < 128 || s->K < 128 || s->N % 128 || s->K % 128 || s->N > (1 << 20) || s->K > (1 << 20)) return SPENSE_ERR_SHAPE;
  const int full = s->split == SPENSE_SPLIT_OUT ? s->N : s->K;
  if (s->n_dense < 0 || s->n_dense > full || s->n_dense % 128) return SPENSE_ERR_SHAPE;
  if (s->split == SPENSE_SPLIT_OUT && (s->N - s->n_dense) % 256) return SPENSE_ERR_SHAPE;
  return SPENSE_OK;
}

int linear_impl(const Launch& L, const spense_linear_shape_t* ls, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t sx_stride,
                int32_t M, void* d_y, int32_t y_dtype, void* d_ws, cudaStream_t stream) {
  const bool in_split = ls->split == SPENSE_SPLIT_IN;
  const Geometry g = make_geometry_linear(ls->N, ls->K, ls->n_dense, in_split);
  const int mode = in_split ? 1 : 2;
  const Plan pl = plan_of(M, L.sms, ls->K, in_split);
  const Schedule& sc = get_schedule(mode, g, pl);
  const uint8_t* section = reinterpret_cast<const uint8_t*>(d_blob) + kBlobHeaderBytes;
  CUtensorMap tm, tws, twd;
  int st = make_tmap(&tm, d_x, ls->K, M, pl.n_pad / 2);
  if (!st) st = make_tmap_section(&tws, section, g.total_bytes - kBlobHeaderBytes, kSparseOperandBytes / 128);
  if (!st) st = make_tmap_section(&twd, section, g.total_bytes - kBlobHeaderBytes, kOperandBytes / 128);
  if (st) return st;
  const spense_shape_t hdr_shape = {g.H, g.I, g.I_d};          // what the header of this blob states
  for (int blk0 = 0; blk0 < pl.nb; blk0 += pl.par) {
    GemmParams p = {};
    fill_common(p, sc, pl, &hdr_shape, d_blob, M, d_ws);
    p.kind = in_split ? kBlobLinearIn : kBlobLinearOut;
    p.nb = pl.nb - blk0 < pl.par ? pl.nb - blk0 : pl.par;
    p.blk0 = blk0;
    p.section = section;
    p.mode = mode;
    if (in_split) {
      p.num_tiles = g.dn_tiles; p.tiles_sparse = 0;
      p.ns = g.dn_ns; p.nd = g.dn_nd; p.dense_k0 = g.I_s;
    } else {
      p.num_tiles = g.gu_tiles; p.tiles_sparse = g.gu_tiles_sparse;
      p.ns = g.gu_ns; p.nd = g.gu_nd; p.dense_k0 = 0;
    }
    p.s_act = d_sx; p.sh_stride = sx_stride;
    p.scale0 = 0; p.scale1 = 0;
    p.y = d_y;
    p.y_dtype = y_dtype;
    p.ld_out = ls->N; p.out_rows = ls->N;
    st = launch_gemm(p, tm, tws, twd, false, L.dev, stream);
    if (st) return st;
  }
  return SPENSE_OK;
}

int linear_entry(int split, const spense_linear_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t sx_stride,
                 int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  int st = check_linear_shape(shape);
  if (st) return st;
  if (shape->split != split || !d_blob || !d_x || !d_sx || !d_y || M < 1 || M > kMaxTokens || (sx_stride != 0 && sx_stride != 1) ||
      (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16) || !d_ws)
    return SPENSE_ERR_ARG;
  if (!aligned(d_blob, 128) || !aligned(d_x, 128) || !aligned(d_y, 16) || !aligned(d_sx, 4) || !aligned(d_ws, 128)) return SPENSE_ERR_ALIGN;
  if (ws_bytes < ws_bytes_for(M)) return SPENSE_ERR_BUFFER_TOO_SMALL;
  Launch L;
  st = check_device(&L.dev, &L.sms);
  if (st) return st;
  st = pending_device_error();
  if (st) return st;
  return linear_impl(L, shape, d_blob, d_x, d_sx, sx_stride, M, d_y, y_dtype, d_ws, reinterpret_cast<cudaStream_t>(stream));
}

int check_ws(const spense_shape_t* shape, int M, const void* d_ws, size_t ws_bytes) {
  if (!d_ws) return SPENSE_ERR_ARG;
  if (!aligned(d_ws, 128)) return SPENSE_ERR_ALIGN;
  size_t need = 0;
  int st = spense_workspace_size(shape, M, &need);
  if (st) return st;
  return ws_bytes < need ? SPENSE_ERR_BUFFER_TOO_SMALL : SPENSE_OK;
}

// what every GEMM entry point does before it launches
int enter(const spense_shape_t* shape, int M, const void* d_ws, size_t ws_bytes, Launch* L) {
  int st = check_ws(shape, M, d_ws, ws_bytes);
  if (st) return st;
  st = check_device(&L->dev, &L->sms);
  if (st) return st;
  return pending_device_error();
}

}  // namespace
}  // namespace spense

using namespace spense;

extern "C" {

int spense_version(void) { return 2; }

#ifdef SPENSE_DEBUG_HOOKS
// debug hook (SPENSE_DEBUG_HOOKS builds only): per-CTA globaltimer timeline, 16 int64 per span, of the next launches
void spense_debug_set_trace(void* d_buf) { g_trace = reinterpret_cast<long long*>(d_buf); }
#endif

const char* spense_strerror(int status) {
  switch (status) {
    case SPENSE_OK: return "ok";
    case SPENSE_ERR_ARG: return "invalid argument";
    case SPENSE_ERR_ALIGN: return "pointer not sufficiently aligned";
    case SPENSE_ERR_SHAPE: return "unsupported shape (H, I, I_dense must be multiples of 128, I_dense <= I)";
    case SPENSE_ERR_BUFFER_TOO_SMALL: return "buffer smaller than the size query";
    case SPENSE_ERR_NOT_2_4: return "a group of 4 in the sparse region has more than 2 non-zeros";
    case SPENSE_ERR_NAN_WEIGHT: return "NaN weight byte (0x7F / 0xFF)";
    case SPENSE_ERR_BAD_PERM: return "perm is not a bijection";
    case SPENSE_ERR_ARCH: return "device is not sm_100 (no fallback path exists)";
    case SPENSE_ERR_CUDA: return "CUDA error";
    case SPENSE_ERR_BAD_BLOB: return "blob header does not match";
    case SPENSE_ERR_TIMEOUT: return "a CTA gave up waiting for the other CTAs of its launch and trapped (device shared with other work?); the CUDA context is lost";
    case SPENSE_ERR_STATIC_SCRATCH: return "request exceeds the built-in scratch of the allocation-free entry point (see its MAX in spense.h)";
    default: return "unknown status";
  }
}

int spense_device_status(int clear) {
  const int st = pending_device_error();
  if (clear && g_status) *reinterpret_cast<volatile int*>(g_status) = 0;
  return st;
}

int spense_schedule(const spense_shape_t* shape, int32_t M, int32_t mode, int32_t sms, int32_t* out_span_begin, int32_t* out_info) {
  int st = check_shape(shape);
  if (st) return st;
  if (M < 1 || M > kMaxTokens || (mode != 0 && mode != 1) || sms < 2 || sms > kMaxSpans || !out_span_begin) return SPENSE_ERR_ARG;
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const Plan pl = plan_of(M, sms, mode == 0 ? g.H : g.I, mode == 1);
  const Schedule& sc = get_schedule(mode, g, pl);
  for (int i = 0; i <= sc.n_spans; ++i) out_span_begin[i] = sc.span_begin[i];
  if (out_info) {
    out_info[0] = sc.span_begin[sc.n_spans];
    out_info[1] = pl.par;
    out_info[2] = pl.n_pad;
    out_info[3] = pl.ring;
    out_info[4] = pl.nb;
    out_info[5] = 2;
  }
  return sc.n_spans;
}

int spense_perm_from_dense_idx(int32_t I, const int32_t* h_dense_idx, int32_t n_dense, int32_t* h_perm) {
  if (I < 0 || n_dense < 0 || n_dense > I || !h_perm || (n_dense && !h_dense_idx)) return SPENSE_ERR_ARG;
  std::vector<uint8_t> is_dense((size_t)I, 0);
  for (int i = 0; i < n_dense; ++i) {
    const int d = h_dense_idx[i];
    if (d < 0 || d >= I || is_dense[d]) return SPENSE_ERR_ARG;
    is_dense[d] = 1;
  }
  int w = 0;
  for (int i = 0; i < I; ++i) if (!is_dense[i]) h_perm[w++] = i;
  for (int i = 0; i < I; ++i) if (is_dense[i]) h_perm[w++] = i;
  return SPENSE_OK;
}

int spense_dense_idx_last(int32_t I, int32_t n_dense, int32_t* h_dense_idx) {
  if (I < 0 || n_dense < 0 || n_dense > I || (n_dense && !h_dense_idx)) return SPENSE_ERR_ARG;
  for (int i = 0; i < n_dense; ++i) h_dense_idx[i] = I - n_dense + i;
  return SPENSE_OK;
}

int spense_pack_sizes(const spense_shape_t* shape, size_t* blob_bytes, size_t* workspace_bytes) {
  int st = check_shape(shape);
  if (st) return st;
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  if (blob_bytes) *blob_bytes = g.total_bytes;
  if (workspace_bytes) *workspace_bytes = 128 + (size_t)shape->I * sizeof(int);
  return SPENSE_OK;
}

int spense_pack(const spense_shape_t* shape, const uint8_t* d_wgate, const uint8_t* d_wup, const uint8_t* d_wdown,
                const float* h_w_scale, const int32_t* d_perm, void* d_blob, size_t blob_bytes,
                const spense_canon_t* canon, void* d_ws, size_t ws_bytes, int64_t* h_err_where, spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_wgate || !d_wup || !d_wdown || !h_w_scale || !d_blob || !d_ws) return SPENSE_ERR_ARG;
  if (!aligned(d_wgate, 128) || !aligned(d_wup, 128) || !aligned(d_wdown, 128) || !aligned(d_blob, 128) ||
      !aligned(d_ws, 128) || (d_perm && !aligned(d_perm, 4)))
    return SPENSE_ERR_ALIGN;
  size_t need_blob = 0, need_ws = 0;
  spense_pack_sizes(shape, &need_blob, &need_ws);
  if (blob_bytes < need_blob || ws_bytes < need_ws) return SPENSE_ERR_BUFFER_TOO_SMALL;
  st = check_device(nullptr, nullptr);
  if (st) return st;
  return launch_pack(shape, d_wgate, d_wup, d_wdown, h_w_scale, d_perm, d_blob, canon, d_ws, h_err_where,
                     reinterpret_cast<cudaStream_t>(stream));
}

int spense_workspace_size(const spense_shape_t* shape, int32_t M, size_t* bytes) {
  int st = check_shape(shape);
  if (st) return st;
  if (M < 1 || M > kMaxTokens || !bytes) return SPENSE_ERR_ARG;
  *bytes = ws_bytes_for(M);
  return SPENSE_OK;
}

int spense_workspace_init(void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  if (!d_ws) return SPENSE_ERR_ARG;
  if (ws_bytes < (size_t)kWsFixedBytes) return SPENSE_ERR_BUFFER_TOO_SMALL;
  // everything the library sets up once per process / device happens here, outside any capture: the pinned status word,
  // the tensor-map encoder entry point, each GEMM kernel's shared-memory opt-in and residency query
  int dev = 0;
  int st = check_device(&dev, nullptr);
  if (st) return st;
  st = prepare_gemm_kernels(dev);
  if (st) return st;
  return cudaMemsetAsync(d_ws, 0, kWsFixedBytes, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

int spense_gate_up(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t M,
                   const float* d_sh, int32_t sh_stride, uint8_t* d_hq, float* d_h_f32, void* d_ws, size_t ws_bytes,
                   spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_blob || !d_x || !d_sx || !d_sh || !d_hq || M < 1 || M > kMaxTokens || (sh_stride != 0 && sh_stride != 1)) return SPENSE_ERR_ARG;
  if (!aligned(d_blob, 128) || !aligned(d_x, 128) || !aligned(d_hq, 16) || !aligned(d_sx, 4) || !aligned(d_sh, 4) ||
      (d_h_f32 && !aligned(d_h_f32, 16)))
    return SPENSE_ERR_ALIGN;
  Launch L;
  st = enter(shape, M, d_ws, ws_bytes, &L);
  if (st) return st;
  return gate_up_impl(L, shape, d_blob, d_x, d_sx, M, d_sh, sh_stride, d_hq, d_h_f32, d_ws, false, false,
                      reinterpret_cast<cudaStream_t>(stream));
}

int spense_down(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_hq, const float* d_sh, int32_t sh_stride,
                int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes, const void* d_next_blob,
                spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_blob || !d_hq || !d_sh || !d_y || M < 1 || M > kMaxTokens || (sh_stride != 0 && sh_stride != 1) ||
      (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16))
    return SPENSE_ERR_ARG;
  if (!aligned(d_blob, 128) || !aligned(d_hq, 128) || !aligned(d_y, 16) || !aligned(d_sh, 4) || !aligned(d_next_blob, 128))
    return SPENSE_ERR_ALIGN;
  Launch L;
  st = enter(shape, M, d_ws, ws_bytes, &L);
  if (st) return st;
  return down_impl(L, shape, d_blob, d_hq, d_sh, sh_stride, M, d_y, y_dtype, d_ws, false, d_next_blob,
                   reinterpret_cast<cudaStream_t>(stream));
}

int spense_mlp(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t M,
               const float* d_sh, int32_t sh_stride, uint8_t* d_hq_scratch, float* d_h_f32, void* d_y, int32_t y_dtype,
               void* d_ws, size_t ws_bytes, const void* d_next_blob, spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_blob || !d_x || !d_sx || !d_sh || !d_hq_scratch || !d_y || M < 1 || M > kMaxTokens || (sh_stride != 0 && sh_stride != 1) ||
      (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16))
    return SPENSE_ERR_ARG;
  if (!aligned(d_blob, 128) || !aligned(d_x, 128) || !aligned(d_hq_scratch, 128) || !aligned(d_y, 16) ||
      !aligned(d_sx, 4) || !aligned(d_sh, 4) || (d_h_f32 && !aligned(d_h_f32, 16)) || !aligned(d_next_blob, 128))
    return SPENSE_ERR_ALIGN;
  Launch L;
  st = enter(shape, M, d_ws, ws_bytes, &L);
  if (st) return st;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  st = gate_up_impl(L, shape, d_blob, d_x, d_sx, M, d_sh, sh_stride, d_hq_scratch, d_h_f32, d_ws, true, true, s);
  if (st) return st;
  return down_impl(L, shape, d_blob, d_hq_scratch, d_sh, sh_stride, M, d_y, y_dtype, d_ws, true, d_next_blob, s);
}

int spense_mlp_dyn(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t M,
                   float* d_sh_out, uint8_t* d_hq_scratch, float* d_h_scratch, void* d_y, int32_t y_dtype, void* d_ws,
                   size_t ws_bytes, const void* d_next_blob, spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_blob || !d_x || !d_sx || !d_sh_out || !d_hq_scratch || !d_h_scratch || !d_y || M < 1 || M > kMaxTokens ||
      (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16))
    return SPENSE_ERR_ARG;
  if (!aligned(d_blob, 128) || !aligned(d_x, 128) || !aligned(d_hq_scratch, 128) || !aligned(d_y, 16) ||
      !aligned(d_sx, 4) || !aligned(d_sh_out, 4) || !aligned(d_h_scratch, 16) || !aligned(d_next_blob, 128))
    return SPENSE_ERR_ALIGN;
  Launch L;
  st = enter(shape, M, d_ws, ws_bytes, &L);
  if (st) return st;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  // gate_up (h in fp32, max|h| per CTA) -> row requant (s_h, Hq), per launch of token blocks; then down
  st = gate_up_impl(L, shape, d_blob, d_x, d_sx, M, d_sx, 0, d_hq_scratch, d_h_scratch, d_ws, true, true, s, true, d_sh_out);
  if (st) return st;
  return down_impl(L, shape, d_blob, d_hq_scratch, d_sh_out, 1, M, d_y, y_dtype, d_ws, true, d_next_blob, s);
}

int spense_mlp_host(const spense_shape_t* shape, const void* d_blob, const uint8_t* h_x, const float* h_sx, int32_t M,
                    const float* h_sh, int32_t sh_stride, void* h_y, int32_t y_dtype, uint8_t* d_x, float* d_scales,
                    uint8_t* d_hq_scratch, void* d_y, void* d_ws, size_t ws_bytes, const void* d_next_blob,
                    spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!h_x || !h_sx || !h_sh || !h_y || !d_x || !d_scales || M < 1 || M > kMaxTokens || (sh_stride != 0 && sh_stride != 1) ||
      (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16))
    return SPENSE_ERR_ARG;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  const size_t n_sh = sh_stride ? (size_t)M : 1;
  if (cudaMemcpyAsync(d_x, h_x, (size_t)M * shape->H, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(d_scales, h_sx, (size_t)M * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(d_scales + M, h_sh, n_sh * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  st = spense_mlp(shape, d_blob, d_x, d_scales, M, d_scales + M, sh_stride, d_hq_scratch, nullptr, d_y, y_dtype, d_ws,
                  ws_bytes, d_next_blob, stream);
  if (st) return st;
  const size_t esz = y_dtype == SPENSE_F32 ? 4 : 2;
  if (cudaMemcpyAsync(h_y, d_y, (size_t)M * shape->H * esz, cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return SPENSE_ERR_CUDA;
  return pending_device_error();
}

int spense_mlp_stack_host(const spense_shape_t* shape, const void* const* d_blobs, int32_t n_layers, const uint8_t* h_x,
                          const float* h_sx, int32_t M, const float* h_sh, int32_t sh_stride, void* h_y, int32_t y_dtype, uint8_t* d_x,
                          float* d_scales, uint8_t* d_hq_scratch, void* d_y, void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_blobs || n_layers < 1 || !h_x || !h_sx || !h_sh || !h_y || !d_x || !d_scales || M < 1 || M > kMaxTokens ||
      (sh_stride != 0 && sh_stride != 1) || (y_dtype != SPENSE_F32 && y_dtype != SPENSE_BF16))
    return SPENSE_ERR_ARG;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  const size_t n_sh = sh_stride ? (size_t)M : 1;
  if (cudaMemcpyAsync(d_x, h_x, (size_t)M * shape->H, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(d_scales, h_sx, (size_t)M * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(d_scales + M, h_sh, n_sh * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  for (int i = 0; i < n_layers; ++i) {
    st = spense_mlp(shape, d_blobs[i], d_x, d_scales, M, d_scales + M, sh_stride, d_hq_scratch, nullptr, d_y, y_dtype, d_ws, ws_bytes,
                    d_blobs[(i + 1) % n_layers], stream);
    if (st) return st;
  }
  const size_t esz = y_dtype == SPENSE_F32 ? 4 : 2;
  if (cudaMemcpyAsync(h_y, d_y, (size_t)M * shape->H * esz, cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return SPENSE_ERR_CUDA;
  return pending_device_error();
}

int spense_linear_pack_sizes(const spense_linear_shape_t* shape, size_t* blob_bytes, size_t* workspace_bytes) {
  int st = check_linear_shape(shape);
  if (st) return st;
  const Geometry g = make_geometry_linear(shape->N, shape->K, shape->n_dense, shape->split == SPENSE_SPLIT_IN);
  if (blob_bytes) *blob_bytes = g.total_bytes;
  const int n_perm = shape->split == SPENSE_SPLIT_IN ? shape->K : shape->N;
  if (workspace_bytes) *workspace_bytes = 128 + (size_t)n_perm * sizeof(int);
  return SPENSE_OK;
}

int spense_pack_linear(const spense_linear_shape_t* shape, const uint8_t* d_w, float w_scale, const int32_t* d_perm, void* d_blob,
                       size_t blob_bytes, const spense_linear_canon_t* canon, void* d_ws, size_t ws_bytes, int64_t* h_err_where,
                       spense_stream_t stream) {
  int st = check_linear_shape(shape);
  if (st) return st;
  if (!d_w || !d_blob || !d_ws) return SPENSE_ERR_ARG;
  if (!aligned(d_w, 128) || !aligned(d_blob, 128) || !aligned(d_ws, 128) || (d_perm && !aligned(d_perm, 4))) return SPENSE_ERR_ALIGN;
  size_t need_blob = 0, need_ws = 0;
  spense_linear_pack_sizes(shape, &need_blob, &need_ws);
  if (blob_bytes < need_blob || ws_bytes < need_ws) return SPENSE_ERR_BUFFER_TOO_SMALL;
  st = check_device(nullptr, nullptr);
  if (st) return st;
  return launch_pack_linear(shape, d_w, w_scale, d_perm, d_blob, canon, d_ws, h_err_where, reinterpret_cast<cudaStream_t>(stream));
}

int spense_linear_workspace_size(const spense_linear_shape_t* shape, int32_t M, size_t* bytes) {
  int st = check_linear_shape(shape);
  if (st) return st;
  if (M < 1 || M > kMaxTokens || !bytes) return SPENSE_ERR_ARG;
  *bytes = ws_bytes_for(M);
  return SPENSE_OK;
}

int spense_linear_out_split(const spense_linear_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t sx_stride,
                            int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  return linear_entry(SPENSE_SPLIT_OUT, shape, d_blob, d_x, d_sx, sx_stride, M, d_y, y_dtype, d_ws, ws_bytes, stream);
}

int spense_linear_in_split(const spense_linear_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx, int32_t sx_stride,
                           int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  return linear_entry(SPENSE_SPLIT_IN, shape, d_blob, d_x, d_sx, sx_stride, M, d_y, y_dtype, d_ws, ws_bytes, stream);
}

int spense_select_workspace_size(const spense_shape_t* shape, size_t* bytes) {
  int st = check_shape(shape);
  if (st) return st;
  if (!bytes) return SPENSE_ERR_ARG;
  // three score vectors, the combined score, the ranks, W_down's column sums per 64-row chunk
  *bytes = (size_t)shape->I * (5 + (size_t)(shape->H + 63) / 64) * sizeof(float) + 128;
  return SPENSE_OK;
}

int spense_select_dense(const spense_shape_t* shape, const float* d_wgate, const float* d_wup, const float* d_wdown,
                        const float* d_hdiag_x, const float* d_hdiag_h, float eps, float* d_score, int32_t* d_dense_idx,
                        int32_t* d_perm, void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_wgate || !d_wup || !d_wdown || !d_hdiag_x || !d_hdiag_h || !d_perm || !d_ws || (shape->I_dense > 0 && !d_dense_idx) ||
      !(eps >= 0.0f))
    return SPENSE_ERR_ARG;
  if (!aligned(d_wgate, 16) || !aligned(d_wup, 16) || !aligned(d_wdown, 16) || !aligned(d_hdiag_x, 16) || !aligned(d_ws, 16))
    return SPENSE_ERR_ALIGN;
  size_t need = 0;
  spense_select_workspace_size(shape, &need);
  if (ws_bytes < need) return SPENSE_ERR_BUFFER_TOO_SMALL;
  st = check_device(nullptr, nullptr);
  if (st) return st;
  return launch_select(shape, d_wgate, d_wup, d_wdown, d_hdiag_x, d_hdiag_h, eps, d_score, d_dense_idx, d_perm, d_ws,
                       reinterpret_cast<cudaStream_t>(stream));
}

int spense_prune_2to4_magnitude(const spense_shape_t* shape, float* d_wgate, float* d_wup, float* d_wdown, const int32_t* d_perm,
                                spense_stream_t stream) {
  int st = check_shape(shape);
  if (st) return st;
  if (!d_wgate || !d_wup || !d_wdown) return SPENSE_ERR_ARG;
  if (!aligned(d_wgate, 16) || !aligned(d_wup, 16) || !aligned(d_wdown, 16) || (d_perm && !aligned(d_perm, 4))) return SPENSE_ERR_ALIGN;
  st = check_device(nullptr, nullptr);
  if (st) return st;
  return launch_prune(shape, d_wgate, d_wup, d_wdown, d_perm, reinterpret_cast<cudaStream_t>(stream));
}

int spense_prune_obs_workspace_size(int32_t N, int32_t K, size_t* bytes) {
  if (N < 1 || K < 4 || K % 4 || N > 65535 * 64 || K > (1 << 20) || !bytes) return SPENSE_ERR_ARG;   // ceil(N / 64) row tiles must fit gridDim.y (65535)
  *bytes = (size_t)N * 128 * sizeof(float);                       // the per-block errors e of every row
  return SPENSE_OK;
}

int spense_prune_obs_2to4(int32_t N, int32_t K, int32_t K_sparse, float* d_w, const float* d_u, void* d_ws, size_t ws_bytes,
                          spense_stream_t stream) {
  size_t need = 0;
  int st = spense_prune_obs_workspace_size(N, K, &need);
  if (st) return st;
  if (K_sparse < 0 || K_sparse > K || K_sparse % 4 || !d_w || !d_u || !d_ws) return SPENSE_ERR_ARG;
  if (!aligned(d_w, 16) || !aligned(d_u, 16) || !aligned(d_ws, 16)) return SPENSE_ERR_ALIGN;
  if (ws_bytes < need) return SPENSE_ERR_BUFFER_TOO_SMALL;
  st = check_device(nullptr, nullptr);
  if (st) return st;
  if (K_sparse == 0) return SPENSE_OK;
  return launch_prune_obs(N, K, K_sparse, d_w, d_u, d_ws, reinterpret_cast<cudaStream_t>(stream));
}

int spense_probe_read(const void* d_buf, size_t bytes, uint32_t* d_sink, spense_stream_t stream) {
  if (!d_buf || !d_sink || bytes < 32768 || bytes % 32768) return SPENSE_ERR_ARG;
  if (!aligned(d_buf, 128) || !aligned(d_sink, 4)) return SPENSE_ERR_ALIGN;
  int sms = 0;
  int st = check_device(nullptr, &sms);
  if (st) return st;
  return launch_read_probe(d_buf, bytes, d_sink, sms, reinterpret_cast<cudaStream_t>(stream));
}

int spense_quantize_e4m3(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out, float* d_scales,
                         void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  if (!d_in || !d_out || !d_scales || !d_ws || rows < 1 || cols < 1 || (mode != SPENSE_PER_TENSOR && mode != SPENSE_PER_ROW))
    return SPENSE_ERR_ARG;
  if (rows > 0x7FFFFFFF) return SPENSE_ERR_SHAPE;
  if (ws_bytes < (size_t)(rows + 1) * 4) return SPENSE_ERR_BUFFER_TOO_SMALL;
  int st = check_device(nullptr, nullptr);
  if (st) return st;
  return launch_quantize(d_in, rows, cols, mode, d_out, d_scales, d_ws, reinterpret_cast<cudaStream_t>(stream));
}

}  // extern "C"
