// C-ABI entry points of libspense (include/spense.h): argument checking, stream-K schedule,
// tensor-map creation and launches.  No device allocation, no synchronisation in the GEMM calls.
#include <cudaTypedefs.h>

#include <cstdlib>
#include <cstring>
#include <deque>
#include <mutex>
#include <vector>

#include "spense_internal.cuh"

namespace spense {
namespace {

int g_num_sms = 0;
int g_arch_ok = -1;
PFN_cuTensorMapEncodeTiled_v12000 g_encode = nullptr;

int check_device() {
  if (g_arch_ok >= 0) return g_arch_ok ? SPENSE_OK : SPENSE_ERR_ARCH;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SPENSE_ERR_CUDA;
  int major = 0, minor = 0;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
  cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (g_num_sms > kMaxSpans) g_num_sms = kMaxSpans;   // persistent CTAs (all token blocks of a launch together) own fix-up slots 0..kMaxSpans-1
  g_arch_ok = (major == 10 && minor == 0) ? 1 : 0;
  if (g_arch_ok) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
      g_arch_ok = -1;
      return SPENSE_ERR_CUDA;
    }
    g_encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  }
  return g_arch_ok ? SPENSE_OK : SPENSE_ERR_ARCH;
}

int check_shape(const spense_shape_t* s) {
  if (!s) return SPENSE_ERR_ARG;
  if (s->H < 128 || s->I < 128 || s->I_dense < 0 || s->I_dense > s->I) return SPENSE_ERR_SHAPE;
  if (s->H % 128 || s->I % 128 || s->I_dense % 128) return SPENSE_ERR_SHAPE;
  if (s->H > (1 << 20) || s->I > (1 << 20)) return SPENSE_ERR_SHAPE;
  return SPENSE_OK;
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }


size_t part_bytes_for(int n_pad, int spans) { return (size_t)spans * 2 * 2 * n_pad * 128 * sizeof(float); }
// control words, flags, max|h| table, tile flags | partials of gate_up | partials of down (they may run concurrently)
size_t ws_bytes_for(int n_pad, int spans) { return kWsFixedBytes + 2 * part_bytes_for(n_pad, spans); }

double env_double(const char* name, double dflt) {
  const char* v = std::getenv(name);
  return v ? std::atof(v) : dflt;
}

// Token columns of one MMA.  Up to 128 tokens: M padded to 16.  More: blocks of 128 tokens; a launch covers nb_par of
// them side by side (grid = nb_par * k_par CTAs, k_par stream-K spans per block), so the CTAs of different blocks read
// the same weight stage at about the same time: one HBM read, the other blocks hit L2.
int block_tokens() { static const int b = (int)env_double("SPENSE_BLOCK_TOKENS", 128.0); return b == 96 ? 96 : 128; }
int n_pad_of(int M) { return M > 128 ? block_tokens() : (M + 15) / 16 * 16; }
int nb_of(int M) { return M > 128 ? (M + block_tokens() - 1) / block_tokens() : 1; }
// how many of `nb` blocks one launch takes: the largest split within 5 % of the best SM occupancy over all rounds
// (every round is a launch with its own start-up and fix-up tail, so fewer rounds win a near tie)
int nb_par_of(int nb, int sms) {
  auto eff = [&](int c) {
    const int rounds = (nb + c - 1) / c, k = sms / c;
    return (double)nb / (rounds * c) * ((double)(c * k) / sms);
  };
  const int cmax = nb < 32 ? (nb < sms ? nb : sms) : (32 < sms ? 32 : sms);
  double best = 0;
  for (int c = 1; c <= cmax; ++c) best = eff(c) > best ? eff(c) : best;
  int pick = 1;
  for (int c = 1; c <= cmax; ++c)
    if (eff(c) >= 0.95 * best) pick = c;
  return pick;
}

// ---- stream-K schedule: cut the stage sequence into n_spans spans of (nearly) equal bytes.
struct Schedule {
  int mode, H, I, I_d, n_pad, sms, fused;
  int n_spans;
  int span_begin[kMaxSpans + 1];
  uint32_t span_off[kMaxSpans];   // byte offset of the span's first stage image inside its section
  uint32_t span_pre[kMaxSpans];   // bytes of the stages the producer issues before anything else (one ring)
  uint32_t span_len[kMaxSpans];   // bytes of the whole span
  double span_cost[kMaxSpans];    // modelled cost of the span (fused: down spans are sized to equalise gate_up + down)
};

int slot_bytes_of(int n_pad) { return kSparseStageBytes + 2 * n_pad * 128; }
int ring_stages_of(int n_pad) {
  const int stages = (kSmemMax - 1024 - 256 - 20 * n_pad) / slot_bytes_of(n_pad);   // barriers + the two scale tables
  return stages > 8 ? 8 : stages;
}
std::mutex g_sched_mu;
std::deque<Schedule> g_sched;   // deque: references handed out stay valid

// fused = schedules of the single-launch MLP kernel (CTA b runs span n-1-b of gate_up AND of down):
//   gate_up: span boundaries are nudged so that no tile is shared by more than two spans where a tile is not
//            much longer than a span (a 3-way tile finishes last and every down span that reads it waits);
//   down   : spans are sized so that gate_up cost + down cost is the same for every CTA.
const Schedule& get_schedule(int mode, const Geometry& g, int n_pad, int sms, bool fused = false) {
  const Schedule* gate = (fused && mode == 1) ? &get_schedule(0, g, n_pad, sms, true) : nullptr;
  std::lock_guard<std::mutex> lk(g_sched_mu);
  for (const Schedule& s : g_sched)
    if (s.mode == mode && s.H == g.H && s.I == g.I && s.I_d == g.I_d && s.n_pad == n_pad && s.sms == sms && s.fused == (int)fused) return s;
  Schedule sc = {};
  sc.mode = mode; sc.H = g.H; sc.I = g.I; sc.I_d = g.I_d; sc.n_pad = n_pad; sc.sms = sms; sc.fused = fused;
  // cost of a stage.  Every CTA keeps the same number of ring slots in flight, so under HBM contention a
  // stage costs one slot latency plus its bytes: measured on B200 (profiles/) a 40 KB sparse stage takes
  // ~1.12x a 32 KB dense one => fixed part ~36 KB-equivalents; activation bytes come from L2 and weigh less.
  static const double fixed = env_double("SPENSE_SCHED_FIXED", 36864.0), gamma = env_double("SPENSE_SCHED_GAMMA", 0.25);
  const double cs = fixed + kSparseStageBytes + gamma * 2.0 * n_pad * 128, cd = fixed + kDenseStageBytes + gamma * 1.0 * n_pad * 128;
  std::vector<double> cost;
  if (mode == 0) {
    cost.insert(cost.end(), (size_t)g.gu_tiles_sparse * g.gu_ns, cs);
    cost.insert(cost.end(), (size_t)(g.gu_tiles - g.gu_tiles_sparse) * g.gu_nd, cd);
  } else {
    for (int t = 0; t < g.dn_tiles; ++t) {
      cost.insert(cost.end(), (size_t)g.dn_ns, cs);
      cost.insert(cost.end(), (size_t)g.dn_nd, cd);
    }
  }
  const int total = (int)cost.size();
  int spans = sms < kMaxSpans ? sms : kMaxSpans;
  if (spans > total) spans = total;
  double sum = 0;
  for (double c : cost) sum += c;
  sc.n_spans = spans;
  // cumulative share of the cost each span should end at: equal, or (fused down) what is left of an equal
  // share of gate_up + down after the CTA's gate_up span
  std::vector<double> cum(spans + 1, 0.0);
  for (int i = 1; i <= spans; ++i) cum[i] = (double)i / spans;
  if (gate && gate->n_spans == spans) {
    double gsum = 0;
    for (int i = 0; i < spans; ++i) gsum += gate->span_cost[i];
    const double share = (gsum + sum) / spans;
    double tot = 0;
    std::vector<double> w(spans);
    for (int i = 0; i < spans; ++i) { w[i] = share - gate->span_cost[i]; if (w[i] < 0.25 * sum / spans) w[i] = 0.25 * sum / spans; tot += w[i]; }
    double run = 0;
    for (int i = 0; i < spans; ++i) { run += w[i]; cum[i + 1] = run / tot; }
  }
  double acc = 0;
  int s = 0;
  sc.span_begin[0] = 0;
  for (int i = 1; i < spans; ++i) {
    const double target = sum * cum[i];
    while (s < total && acc + 0.5 * cost[s] < target) acc += cost[s++];
    int b = s;
    if (b <= sc.span_begin[i - 1]) b = sc.span_begin[i - 1] + 1;     // every span owns >= 1 stage
    if (b > total - (spans - i)) b = total - (spans - i);
    while (s < b) acc += cost[s++];
    sc.span_begin[i] = b;
  }
  sc.span_begin[spans] = total;
  if (fused && mode == 0) {
    // a span lying strictly inside a tile makes the tile 3-way: stretch it to the nearer tile boundary
    int tf = 0;
    for (int t = 0; t < g.gu_tiles; ++t) {
      const int per = t < g.gu_tiles_sparse ? g.gu_ns : g.gu_nd;
      const int te = tf + per;
      if (per < 2 * total / spans) {
        for (int m = 1; m + 1 < spans; ++m) {
          if (sc.span_begin[m] > tf && sc.span_begin[m + 1] < te) {
            const int head = sc.span_begin[m] - tf, tail = te - sc.span_begin[m + 1];
            if (head <= tail && sc.span_begin[m - 1] < tf) sc.span_begin[m] = tf;
            else if (sc.span_begin[m + 2] > te) sc.span_begin[m + 1] = te;
            else if (sc.span_begin[m - 1] < tf) sc.span_begin[m] = tf;
          }
        }
      }
      tf = te;
    }
  }
  for (int i = 0; i < spans; ++i) {
    double c = 0;
    for (int k = sc.span_begin[i]; k < sc.span_begin[i + 1]; ++k) c += cost[k];
    sc.span_cost[i] = c;
  }
  // byte offsets: the blob stores the stage images in exactly this linear order
  std::vector<uint32_t> bytes(total);
  if (mode == 0) {
    for (int i = 0; i < total; ++i) bytes[i] = i < g.gu_tiles_sparse * g.gu_ns ? kSparseStageBytes : kDenseStageBytes;
  } else {
    const int per = g.dn_ns + g.dn_nd;
    for (int i = 0; i < total; ++i) bytes[i] = (i % per) < g.dn_ns ? kSparseStageBytes : kDenseStageBytes;
  }
  const int ring = ring_stages_of(n_pad);
  uint64_t off = 0;
  int st = 0;
  for (int i = 0; i < spans; ++i) {
    while (st < sc.span_begin[i]) off += bytes[st++];
    sc.span_off[i] = (uint32_t)off;
    uint32_t pre = 0;
    for (int k = sc.span_begin[i]; k < sc.span_begin[i + 1] && k < sc.span_begin[i] + ring; ++k) pre += bytes[k];
    sc.span_pre[i] = pre;
    uint32_t len = 0;
    for (int k = sc.span_begin[i]; k < sc.span_begin[i + 1]; ++k) len += bytes[k];
    sc.span_len[i] = len;
  }
  g_sched.push_back(sc);
  return g_sched.back();
}

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

// header cache: one D2H copy per (blob pointer), so the GEMM calls stay asynchronous afterwards
struct HeaderEntry { const void* p; BlobHeader h; };
std::mutex g_hdr_mu;
std::vector<HeaderEntry> g_hdr_cache;

void forget_header(const void* d_blob) {
  std::lock_guard<std::mutex> lk(g_hdr_mu);
  for (size_t i = 0; i < g_hdr_cache.size(); ++i)
    if (g_hdr_cache[i].p == d_blob) { g_hdr_cache.erase(g_hdr_cache.begin() + i); break; }
}

int read_header(const void* d_blob, const spense_shape_t* shape, BlobHeader* out) {
  std::mutex& mu = g_hdr_mu;
  std::vector<HeaderEntry>& cache = g_hdr_cache;
  using Entry = HeaderEntry;
  {
    std::lock_guard<std::mutex> lk(mu);
    for (const Entry& e : cache)
      if (e.p == d_blob && e.h.H == shape->H && e.h.I == shape->I && e.h.I_dense == shape->I_dense) { *out = e.h; return SPENSE_OK; }
  }
  BlobHeader h;
  if (cudaMemcpy(&h, d_blob, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (h.magic != kBlobMagic || h.version != kBlobVersion || h.H != shape->H || h.I != shape->I || h.I_dense != shape->I_dense)
    return SPENSE_ERR_BAD_BLOB;
  std::lock_guard<std::mutex> lk(mu);
  for (Entry& e : cache)
    if (e.p == d_blob) { e.h = h; *out = h; return SPENSE_OK; }
  cache.push_back({d_blob, h});
  *out = h;
  return SPENSE_OK;
}

// bytes of span k that the PREVIOUS launch pulls into L2 during its tail: at least one ring
uint32_t next_prefetch_bytes(const Schedule& sc, int k) {
  static const uint32_t want = (uint32_t)(env_double("SPENSE_PF_NEXT_KB", 640.0) * 1024.0);
  uint32_t n = sc.span_pre[k] > want ? sc.span_pre[k] : want;
  return n < sc.span_len[k] ? n : sc.span_len[k];
}

int g_fused = -1;               // spense_mlp as ONE persistent launch (SPENSE_FUSED / spense_debug_set_fused); -1 = read the environment
long long* g_trace = nullptr;   // debug: set by spense_debug_set_trace (not part of the public ABI)

void fill_common(GemmParams& p, const Schedule& sc, int M, int n_pad, void* d_ws) {
  p.trace = g_trace;
  if (g_trace) g_trace += (size_t)kMaxSpans * 16;   // debug: consecutive launches fill consecutive timelines
  p.n_spans = sc.n_spans;
  std::memcpy(p.span_begin, sc.span_begin, sizeof(int) * (sc.n_spans + 1));
  static const uint32_t self_want = (uint32_t)(env_double("SPENSE_PF_SELF_KB", 160.0) * 1024.0);
  for (int i = 0; i < sc.n_spans; ++i) {                    // own stages pulled into L2 while waiting for the previous kernel
    const uint32_t from = next_prefetch_bytes(sc, i);
    const uint32_t left = sc.span_len[i] - from;
    p.self_off[i] = from - sc.span_pre[i];
    p.self_len[i] = self_want < left ? self_want : left;
  }
  p.nb = 1;
  p.blk0 = 0;
  p.M = M;
  p.n_pad = n_pad;
  p.slot_bytes = slot_bytes_of(n_pad);
  p.num_stages = ring_stages_of(n_pad);
  p.acc_stride = n_pad <= 32 ? 32 : (n_pad <= 64 ? 64 : (n_pad <= 96 ? 96 : (n_pad <= 112 ? 112 : 128)));
  p.num_acc_bufs = n_pad <= 112 ? 2 : 1;                    // 2 buffers x 2 accumulators x 112 columns = 448, metadata at 480
  // separate launches run one after the other and share the control words, flags and partial slots (the
  // partials then stay hot in L2); the fused kernel gives its down phase the second set (use_second_ws_half)
  uint8_t* ws = reinterpret_cast<uint8_t*>(d_ws);
  p.ws_ctrl = reinterpret_cast<int*>(ws);
  p.flags = reinterpret_cast<int*>(ws + 128);
  p.partials = reinterpret_cast<float*>(ws + kWsFixedBytes);
}

void use_second_ws_half(GemmParams& p, void* d_ws) {
  uint8_t* ws = reinterpret_cast<uint8_t*>(d_ws);
  p.ws_ctrl = reinterpret_cast<int*>(ws) + 2;
  p.flags = reinterpret_cast<int*>(ws + 128 + kMaxSpans * 2 * sizeof(int));
  p.partials = reinterpret_cast<float*>(ws + kWsFixedBytes + part_bytes_for(p.n_pad, kMaxSpans));
}

// L2 prefetch hint: while this launch runs its fix-up tail, pull what the next launch streams first.
void fill_next(GemmParams& p, const uint8_t* next_section, const Schedule& next) {
  static const bool enabled = env_double("SPENSE_L2_PREFETCH", 1.0) != 0.0;
  if (!enabled || !next_section) return;
  p.next_base = next_section;
  static const int pace = (int)env_double("SPENSE_PF_PACE_NS", 750.0);
  p.pf_pace_ns = pace;
  for (int i = 0; i < p.n_spans; ++i) {
    const int k = i < next.n_spans ? i : next.n_spans - 1;
    p.next_off[i] = next.span_off[k];
    p.next_len[i] = i < next.n_spans ? next_prefetch_bytes(next, k) : 0;
  }
}

// parameter block + tensor map of one gate_up launch over tokens [m0, m0 + Mb)
int gate_up_params(const Geometry& g, const BlobHeader& hdr, const void* d_blob, const uint8_t* d_x, const float* d_sx,
                   int m0, int Mb, const float* d_sh, int32_t sh_stride, uint8_t* d_hq, float* d_h_f32, void* d_ws,
                   bool dynamic, GemmParams& p, CUtensorMap& tm, bool fused = false, int k_par = 0, int nb_launch = 1,
                   int blk0 = 0) {
  const int n_pad = n_pad_of(Mb);
  const Schedule& sc = get_schedule(0, g, n_pad, k_par > 0 ? k_par : g_num_sms, fused);
  p = GemmParams{};
  fill_common(p, sc, Mb, n_pad, d_ws);
  p.nb = nb_launch; p.blk0 = blk0;
  p.section = reinterpret_cast<const uint8_t*>(d_blob) + hdr.gate_up_off;
  p.mode = 0;
  p.num_tiles = g.gu_tiles; p.tiles_sparse = g.gu_tiles_sparse;
  p.ns = g.gu_ns; p.nd = g.gu_nd; p.dense_k0 = 0;
  p.s_act = d_sx + m0;
  p.s_h = d_sh + (size_t)m0 * sh_stride; p.sh_stride = sh_stride;
  p.w_scale0 = hdr.w_scale[0]; p.w_scale1 = hdr.w_scale[1];
  p.hq = d_hq + (size_t)m0 * g.I;
  p.h_f32 = d_h_f32 ? d_h_f32 + (size_t)m0 * g.I : nullptr;
  p.amax_part = dynamic ? reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(d_ws) + kFlagBytes) : nullptr;
  p.ld_out = g.I; p.out_rows = g.I;
  return make_tmap(&tm, d_x + (size_t)m0 * g.H, g.H, Mb, n_pad);
}

int down_params(const Geometry& g, const BlobHeader& hdr, const void* d_blob, const uint8_t* d_hq, const float* d_sh,
                int32_t sh_stride, int m0, int Mb, void* d_y, int32_t y_dtype, void* d_ws, GemmParams& p, CUtensorMap& tm,
                bool fused = false, int k_par = 0, int nb_launch = 1, int blk0 = 0) {
  const size_t esz = y_dtype == SPENSE_F32 ? 4 : 2;
  const int n_pad = n_pad_of(Mb);
  const Schedule& sc = get_schedule(1, g, n_pad, k_par > 0 ? k_par : g_num_sms, fused);
  p = GemmParams{};
  fill_common(p, sc, Mb, n_pad, d_ws);
  p.nb = nb_launch; p.blk0 = blk0;
  p.section = reinterpret_cast<const uint8_t*>(d_blob) + hdr.down_off;
  p.mode = 1;
  p.num_tiles = g.dn_tiles; p.tiles_sparse = 0;
  p.ns = g.dn_ns; p.nd = g.dn_nd; p.dense_k0 = g.I_s;
  p.s_act = d_sh + (size_t)m0 * sh_stride; p.sh_stride = sh_stride;
  p.w_scale0 = hdr.w_scale[2]; p.w_scale1 = hdr.w_scale[2];
  p.y = reinterpret_cast<uint8_t*>(d_y) + (size_t)m0 * g.H * esz;
  p.y_dtype = y_dtype;
  p.ld_out = g.H; p.out_rows = g.H;
  return make_tmap(&tm, d_hq + (size_t)m0 * g.I, g.I, Mb, n_pad);
}

int gate_up_impl(const spense_shape_t* shape, const BlobHeader& hdr, const void* d_blob, const uint8_t* d_x,
                 const float* d_sx, int32_t M, const float* d_sh, int32_t sh_stride, uint8_t* d_hq, float* d_h_f32,
                 void* d_ws, bool pdl, bool down_follows, cudaStream_t stream, bool dynamic = false) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const int nb = nb_of(M), par = nb_par_of(nb, g_num_sms);
  for (int blk0 = 0; blk0 < nb; blk0 += par) {               // M <= 128: one launch of one block
    const int nb_l = nb - blk0 < par ? nb - blk0 : par;
    GemmParams p;
    CUtensorMap tm;
    int st = gate_up_params(g, hdr, d_blob, d_x, d_sx, 0, M, d_sh, sh_stride, d_hq, d_h_f32, d_ws, dynamic, p, tm, false,
                            g_num_sms / nb_l, nb_l, blk0);
    if (st) return st;
    if (down_follows && nb == 1)                             // the same layer's down projection streams next
      fill_next(p, reinterpret_cast<const uint8_t*>(d_blob) + hdr.down_off, get_schedule(1, g, n_pad_of(M), g_num_sms));
    st = launch_gemm(p, tm, pdl, stream);
    if (st) return st;
  }
  return SPENSE_OK;
}

int down_impl(const spense_shape_t* shape, const BlobHeader& hdr, const void* d_blob, const uint8_t* d_hq,
              const float* d_sh, int32_t sh_stride, int32_t M, void* d_y, int32_t y_dtype, void* d_ws, bool pdl,
              const void* d_next_blob, cudaStream_t stream) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const int nb = nb_of(M), par = nb_par_of(nb, g_num_sms);
  for (int blk0 = 0; blk0 < nb; blk0 += par) {
    const int nb_l = nb - blk0 < par ? nb - blk0 : par;
    GemmParams p;
    CUtensorMap tm;
    int st = down_params(g, hdr, d_blob, d_hq, d_sh, sh_stride, 0, M, d_y, y_dtype, d_ws, p, tm, false, g_num_sms / nb_l, nb_l, blk0);
    if (st) return st;
    if (d_next_blob && nb == 1)                              // the next layer's gate/up weights stream next
      fill_next(p, reinterpret_cast<const uint8_t*>(d_next_blob) + hdr.gate_up_off, get_schedule(0, g, n_pad_of(M), g_num_sms));
    st = launch_gemm(p, tm, pdl, stream);
    if (st) return st;
  }
  return SPENSE_OK;
}

// One token block: gate_up and down as ONE persistent launch (spense_mlp_kernel); down's Hq loads are gated per
// 128-column tile by flags gate_up publishes, no grid-wide barrier in between.
int mlp_fused_impl(const spense_shape_t* shape, const BlobHeader& hdr, const void* d_blob, const uint8_t* d_x,
                   const float* d_sx, int32_t M, const float* d_sh, int32_t sh_stride, uint8_t* d_hq, float* d_h_f32,
                   void* d_y, int32_t y_dtype, void* d_ws, const void* d_next_blob, cudaStream_t stream) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  GemmParams pg, pd;
  CUtensorMap tx, th;
  int st = gate_up_params(g, hdr, d_blob, d_x, d_sx, 0, M, d_sh, sh_stride, d_hq, d_h_f32, d_ws, false, pg, tx, true);
  if (st) return st;
  st = down_params(g, hdr, d_blob, d_hq, d_sh, sh_stride, 0, M, d_y, y_dtype, d_ws, pd, th, true);
  if (st) return st;
  use_second_ws_half(pd, d_ws);
  int* dep = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(d_ws) + kFlagBytes + kAmaxBytes);
  pg.tile_flags = dep;
  pg.tile_cnt = dep + kDepInts;
  pd.dep_flags = dep;
  pd.dep_done = reinterpret_cast<int*>(d_ws) + kCtrlDepDone;
  pd.dep_tiles = g.gu_tiles;
  { static const uint32_t pfb = (uint32_t)(env_double("SPENSE_PF_GATED_KB", 256.0) * 1024.0); pd.gated_pf_bytes = pfb; }
  if (d_next_blob)                                           // the next layer's gate/up weights stream next
    fill_next(pd, reinterpret_cast<const uint8_t*>(d_next_blob) + hdr.gate_up_off, get_schedule(0, g, n_pad_of(M), g_num_sms, true));
  return launch_mlp(pg, tx, pd, th, stream);
}

int check_ws(const spense_shape_t* shape, int M, const void* d_ws, size_t ws_bytes) {
  if (!d_ws) return SPENSE_ERR_ARG;
  if (!aligned(d_ws, 128)) return SPENSE_ERR_ALIGN;
  size_t need = 0;
  int st = spense_workspace_size(shape, M, &need);
  if (st) return st;
  return ws_bytes < need ? SPENSE_ERR_BUFFER_TOO_SMALL : SPENSE_OK;
}

}  // namespace
}  // namespace spense

using namespace spense;

extern "C" {

int spense_version(void) { return 100 * 0 + 1; }

// debug hook (undeclared in spense.h): run spense_mlp (M <= 128) as the fused single-launch kernel (1) or as two
// PDL-chained launches (0, the default: measured 55.5 vs 57.4 us/layer at M=64)
void spense_debug_set_fused(int on) { g_fused = on ? 1 : 0; }

// debug hook (undeclared in spense.h; host only, no device needed): the stream-K schedule the library would use
// for (shape, M, mode 0 gate_up / 1 down, fused, sms).  Writes n_spans + 1 span boundaries (linear stage indices)
// into out_span_begin (room for 161 ints) and returns n_spans, or a negative status.  out_info[0..3] = total
// stages, token blocks per launch, token columns per MMA, ring slots.
int spense_debug_schedule(const spense_shape_t* shape, int32_t M, int32_t mode, int32_t fused, int32_t sms,
                          int32_t* out_span_begin, int32_t* out_info) {
  int st = check_shape(shape);
  if (st) return st;
  if (M < 1 || M > kMaxTokens || (mode != 0 && mode != 1) || sms < 1 || !out_span_begin) return SPENSE_ERR_ARG;
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const int n_pad = n_pad_of(M), nb = nb_of(M), par = nb_par_of(nb, sms);
  const Schedule& sc = get_schedule(mode, g, n_pad, sms / par, fused != 0 && nb == 1);
  for (int i = 0; i <= sc.n_spans; ++i) out_span_begin[i] = sc.span_begin[i];
  if (out_info) {
    out_info[0] = sc.span_begin[sc.n_spans];
    out_info[1] = par;                                       // token blocks side by side in one launch
    out_info[2] = n_pad;
    out_info[3] = ring_stages_of(n_pad);
  }
  return sc.n_spans;
}

// debug hook (undeclared in spense.h): per-CTA globaltimer timeline, 16 int64 per span, of the next launches
void spense_debug_set_trace(void* d_buf) { g_trace = reinterpret_cast<long long*>(d_buf); }

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
    default: return "unknown status";
  }
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
  st = check_device();
  if (st) return st;
  forget_header(d_blob);
  return launch_pack(shape, d_wgate, d_wup, d_wdown, h_w_scale, d_perm, d_blob, canon, d_ws, h_err_where,
                     reinterpret_cast<cudaStream_t>(stream));
}

int spense_workspace_size(const spense_shape_t* shape, int32_t M, size_t* bytes) {
  int st = check_shape(shape);
  if (st) return st;
  if (M < 1 || M > kMaxTokens || !bytes) return SPENSE_ERR_ARG;
  *bytes = ws_bytes_for(M > 128 ? 128 : n_pad_of(M), kMaxSpans);
  return SPENSE_OK;
}

int spense_workspace_init(void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  if (!d_ws) return SPENSE_ERR_ARG;
  if (ws_bytes < (size_t)kWsFixedBytes) return SPENSE_ERR_BUFFER_TOO_SMALL;
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
  st = check_ws(shape, M, d_ws, ws_bytes);
  if (st) return st;
  st = check_device();
  if (st) return st;
  BlobHeader hdr;
  st = read_header(d_blob, shape, &hdr);
  if (st) return st;
  return gate_up_impl(shape, hdr, d_blob, d_x, d_sx, M, d_sh, sh_stride, d_hq, d_h_f32, d_ws, false, false,
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
  st = check_ws(shape, M, d_ws, ws_bytes);
  if (st) return st;
  st = check_device();
  if (st) return st;
  BlobHeader hdr;
  st = read_header(d_blob, shape, &hdr);
  if (st) return st;
  return down_impl(shape, hdr, d_blob, d_hq, d_sh, sh_stride, M, d_y, y_dtype, d_ws, false, d_next_blob,
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
  st = check_ws(shape, M, d_ws, ws_bytes);
  if (st) return st;
  st = check_device();
  if (st) return st;
  BlobHeader hdr;
  st = read_header(d_blob, shape, &hdr);
  if (st) return st;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  if (g_fused < 0) g_fused = env_double("SPENSE_FUSED", 0.0) != 0.0 ? 1 : 0;
  if (g_fused && M <= 128)
    return mlp_fused_impl(shape, hdr, d_blob, d_x, d_sx, M, d_sh, sh_stride, d_hq_scratch, d_h_f32, d_y, y_dtype, d_ws,
                          d_next_blob, s);
  st = gate_up_impl(shape, hdr, d_blob, d_x, d_sx, M, d_sh, sh_stride, d_hq_scratch, d_h_f32, d_ws, true, true, s);
  if (st) return st;
  return down_impl(shape, hdr, d_blob, d_hq_scratch, d_sh, sh_stride, M, d_y, y_dtype, d_ws, true, d_next_blob, s);
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
  st = check_ws(shape, M, d_ws, ws_bytes);
  if (st) return st;
  st = check_device();
  if (st) return st;
  BlobHeader hdr;
  st = read_header(d_blob, shape, &hdr);
  if (st) return st;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  const float* amax = reinterpret_cast<const float*>(reinterpret_cast<const uint8_t*>(d_ws) + kFlagBytes);
  for (int m0 = 0; m0 < M; m0 += 128) {                      // gate_up (h in fp32, max|h| per CTA) -> requant, per token block
    const int Mb = (M - m0) < 128 ? (M - m0) : 128;
    const int n_pad = n_pad_of(Mb);
    st = gate_up_impl(shape, hdr, d_blob, d_x + (size_t)m0 * g.H, d_sx + m0, Mb, d_sx, 0, d_hq_scratch + (size_t)m0 * g.I,
                      d_h_scratch + (size_t)m0 * g.I, d_ws, true, m0 + 128 >= M, s, true);
    if (st) return st;
    const Schedule& sc = get_schedule(0, g, n_pad, g_num_sms);
    st = launch_requant_rows(d_h_scratch + (size_t)m0 * g.I, Mb, g.I, amax, sc.n_spans, n_pad, d_hq_scratch + (size_t)m0 * g.I,
                             d_sh_out + m0, s);
    if (st) return st;
  }
  return down_impl(shape, hdr, d_blob, d_hq_scratch, d_sh_out, 1, M, d_y, y_dtype, d_ws, true, d_next_blob, s);
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
  return cudaStreamSynchronize(s) == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
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
  st = check_device();
  if (st) return st;
  return launch_select(shape, d_wgate, d_wup, d_wdown, d_hdiag_x, d_hdiag_h, eps, d_score, d_dense_idx, d_perm, d_ws,
                       reinterpret_cast<cudaStream_t>(stream));
}

int spense_quantize_e4m3(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out, float* d_scales,
                         void* d_ws, size_t ws_bytes, spense_stream_t stream) {
  if (!d_in || !d_out || !d_scales || !d_ws || rows < 1 || cols < 1 || (mode != SPENSE_PER_TENSOR && mode != SPENSE_PER_ROW))
    return SPENSE_ERR_ARG;
  if (rows > 0x7FFFFFFF) return SPENSE_ERR_SHAPE;
  if (ws_bytes < (size_t)(rows + 1) * 4) return SPENSE_ERR_BUFFER_TOO_SMALL;
  int st = check_device();
  if (st) return st;
  return launch_quantize(d_in, rows, cols, mode, d_out, d_scales, d_ws, reinterpret_cast<cudaStream_t>(stream));
}

}  // extern "C"
