// Host side of the C ABI in include/af.h: ring bookkeeping + validation (a0, a9), tensor-map cache, workspace carve
// and the launch sequence of Algorithm 2 per layer.  Links only libcudart; the driver's
// cuTensorMapEncodeTiled is fetched through cudaGetDriverEntryPoint.  No CPU fallback: every step is a kernel.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <vector>

#include "../../include/af_debug.h"

namespace af { constexpr int AF_MAX_SEGS_K = AF_MAX_SEGS; }
#include "gemm_tcgen05.cuh"
#include "chain.cuh"
#include "elementwise.cuh"

using namespace af;

// ------------------------------------------------------------------------------------------------ errors
static thread_local std::string g_err;
static int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}
#define CUDA_TRY(expr)                                                                              \
  do {                                                                                              \
    cudaError_t e_ = (expr);                                                                        \
    if (e_ != cudaSuccess) return fail(AF_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

static std::atomic<int64_t> g_launches{0};
static int check_launch(const char* what) {
  g_launches.fetch_add(1, std::memory_order_relaxed);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(AF_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
  return AF_OK;
}

// ------------------------------------------------------------------------------------------------ per-kernel timing
// Optional CUDA-event timing of every launch, by kernel class, on the launching stream (bench.py's roofline leg).
enum ProfCat { PC_GEMM_QKV = 0, PC_GEMM_O, PC_GEMM_GATEUP, PC_GEMM_DOWN, PC_GEMM_LM, PC_ATTENTION, PC_ROPE_APPEND,
               PC_RMSNORM, PC_CHAIN, PC_OTHER, PC_COUNT };
struct ProfRec { cudaEvent_t a, b; int cat; };
static bool g_prof_on = false;
static bool g_prof_stages = false;   // af_debug_profile(2): time the per-stage path (one kernel per stage) instead of the layer chain
static std::vector<ProfRec> g_prof;
struct ProfScope {
  cudaStream_t st; ProfRec r; bool on;
  ProfScope(int cat, cudaStream_t s) : st(s), on(g_prof_on) {
    if (!on) return;
    r.cat = cat; cudaEventCreate(&r.a); cudaEventCreate(&r.b); cudaEventRecord(r.a, st);
  }
  ~ProfScope() { if (on) { cudaEventRecord(r.b, st); g_prof.push_back(r); } }
};
static int g_att_mode = 0;   // af_debug_attention: 0 automatic, 1 attention_kernel (mma.sync) always, 2 the units of attention_umma.cuh wherever they apply
extern "C" int af_debug_attention(int mode) {
  if (mode < 0 || mode > 2) return fail(AF_ERR_ARG, "af_debug_attention: mode %d outside [0,2]", mode);
  g_att_mode = mode;
  return AF_OK;
}
extern "C" int af_debug_profile(int enable) { g_prof_on = enable != 0; g_prof_stages = enable == 2; return AF_OK; }
extern "C" int af_debug_profile_read(double* ms_sum, int64_t* counts, int32_t n) {
  if (!ms_sum || !counts || n < PC_COUNT) return fail(AF_ERR_ARG, "need %d slots", (int)PC_COUNT);
  CUDA_TRY(cudaDeviceSynchronize());
  for (int i = 0; i < n; ++i) { ms_sum[i] = 0; counts[i] = 0; }
  for (auto& r : g_prof) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, r.a, r.b);
    ms_sum[r.cat] += ms; counts[r.cat] += 1;
    cudaEventDestroy(r.a); cudaEventDestroy(r.b);
  }
  g_prof.clear();
  return AF_OK;
}

// ------------------------------------------------------------------------------------------------ tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static std::mutex g_mu;
static EncodeTiledFn g_encode = nullptr;
struct MapKey {
  const void* ptr; int elem; unsigned long long d[3], st[2]; unsigned b[3]; int rank, swz;
  bool operator<(const MapKey& o) const { return memcmp(this, &o, sizeof(MapKey)) < 0; }
};
static std::map<MapKey, CUtensorMap> g_maps;

// Cached cuTensorMapEncodeTiled.  dims / box innermost first; strides (bytes) of dims 1..rank-1.
static int get_map_nd(const void* ptr, int elem_bytes, int rank, /* elem_bytes: 2 = bf16, -2 = fp16, 4 = fp32, 1 = uint8 (E4M3 codes) */ const unsigned long long* dims,
                      const unsigned long long* strides, const unsigned* box, int swizzle /* 0 none, 128, 64 or 32 bytes */, CUtensorMap* out) {
  std::lock_guard<std::mutex> lk(g_mu);
  MapKey key;
  memset(&key, 0, sizeof key);
  key.ptr = ptr; key.elem = elem_bytes; key.rank = rank; key.swz = swizzle;
  for (int i = 0; i < rank; ++i) { key.d[i] = dims[i]; key.b[i] = box[i]; }
  for (int i = 0; i + 1 < rank; ++i) key.st[i] = strides[i];
  auto it = g_maps.find(key);
  if (it != g_maps.end()) { *out = it->second; return AF_OK; }
  if (!g_encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(AF_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    g_encode = reinterpret_cast<EncodeTiledFn>(fn);
  }
  if (reinterpret_cast<uintptr_t>(ptr) & 15) return fail(AF_ERR_ARG, "matrix %p must be 16-byte aligned", ptr);
  for (int i = 0; i + 1 < rank; ++i)
    if (strides[i] % 16) return fail(AF_ERR_ARG, "matrix %p: stride %llu is not a multiple of 16 bytes", ptr, strides[i]);
  CUtensorMap m;
  cuuint64_t d[3], st[2];
  cuuint32_t bx[3], estr[3] = {1, 1, 1};
  for (int i = 0; i < rank; ++i) { d[i] = dims[i]; bx[i] = box[i]; }
  for (int i = 0; i + 1 < rank; ++i) st[i] = strides[i];
  const CUtensorMapDataType dt = elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                 : (elem_bytes == -2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16
                                 : (elem_bytes == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32));
  CUresult r = g_encode(&m, dt, rank, const_cast<void*>(ptr), d, st, bx, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        swizzle == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                        : swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                        : swizzle == 32 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(AF_ERR_CUDA, "cuTensorMapEncodeTiled(%p, rank %d) -> %d", ptr, rank, (int)r);
  if (g_maps.size() > 8192) g_maps.clear();
  g_maps[key] = m;
  *out = m;
  return AF_OK;
}

// bf16 row-major [rows, cols] operand matrix, box = [box_rows, 64 cols], 128-byte swizzle, zero fill out of bounds.
static int get_map(const void* ptr, int rows, int cols, int box_rows, CUtensorMap* out, bool fp16 = false) {
  if (cols % 8) return fail(AF_ERR_ARG, "matrix %p [%d,%d] needs a 16-byte row pitch", ptr, rows, cols);
  const unsigned long long dims[2] = {static_cast<unsigned long long>(cols), static_cast<unsigned long long>(rows)};
  const unsigned long long strides[1] = {static_cast<unsigned long long>(cols) * 2};
  const unsigned box[2] = {static_cast<unsigned>(GEMM_BK), static_cast<unsigned>(box_rows)};
  return get_map_nd(ptr, fp16 ? -2 : 2, 2, dims, strides, box, 128, out);
}

// E4M3 weight matrix [rows, cols] (one byte per element), box = [128 rows, 64 codes], no swizzle (the tile is widened to
// the fp16 UMMA layout by the kernel), zero fill out of bounds.
static int get_map_fp8(const void* ptr, int rows, int cols, CUtensorMap* out) {
  if (cols % 16) return fail(AF_ERR_ARG, "FP8 matrix %p [%d,%d] needs a 16-byte row pitch", ptr, rows, cols);
  const unsigned long long dims[2] = {static_cast<unsigned long long>(cols), static_cast<unsigned long long>(rows)};
  const unsigned long long strides[1] = {static_cast<unsigned long long>(cols)};
  const unsigned box[2] = {static_cast<unsigned>(GEMM_BK), static_cast<unsigned>(GEMM_BM)};
  return get_map_nd(ptr, 1, 2, dims, strides, box, 0, out);
}

// Output view of a GEMM (see GemmParams): element (feature f, middle m, token t) at ptr + t*ld_tok + m*ld_mid + f.
struct OutView { void* ptr; int elem_bytes; /* 4 = fp32, 2 = bf16, -2 = fp16 */ int features, n_mid, tokens; long long ld_mid, ld_tok; int box_feat; };
static int get_out_map(const OutView& o, int stg_bytes, CUtensorMap* out) {
  const unsigned long long dims[3] = {static_cast<unsigned long long>(o.features), static_cast<unsigned long long>(o.n_mid),
                                      static_cast<unsigned long long>(o.tokens)};
  const int eb = o.elem_bytes < 0 ? -o.elem_bytes : o.elem_bytes;
  const unsigned long long strides[2] = {static_cast<unsigned long long>(o.ld_mid) * eb,
                                         static_cast<unsigned long long>(o.ld_tok) * eb};
  const int et = o.elem_bytes;
  const unsigned box[3] = {static_cast<unsigned>(o.box_feat), 1u, (o.elem_bytes == 4 && stg_bytes < 4096) ? 16u : 32u};
  // fp16 boxes are staged by stmatrix in the swizzle of their row length (32 features = 64 bytes, 16 = 32 bytes)
  return get_map_nd(o.ptr, et, 3, dims, strides, box, eb == 2 ? o.box_feat * 2 : 0, out);
}

// ------------------------------------------------------------------------------------------------ launches
// Every kernel of the step is launched with programmatic dependent launch: its prologue (barrier init, TMEM
// allocation, tensor-map prefetch, the first weight tiles) overlaps the previous kernel's tail, and each kernel
// executes griddepcontrol.wait before it touches anything the previous kernel wrote.
// Tuning constants (each was an environment knob while it was being measured on B200; DESIGN.md 6.1 has the numbers):
constexpr int kWeightStagesBeforeWait = 3;   // weight stages a GEMM requests before griddepcontrol.wait: 3 beats all 6 by 0.6 %
                                             // (a resident CTA's prefetch competes for HBM with the tail of the kernel it waits for)
constexpr int kMinStages = 5;                // fp32-output GEMMs shrink their epilogue staging until the ring has this many stages
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, int cluster, Args... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[2];
  int n = 0;
  at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[n].val.programmaticStreamSerializationAllowed = 1;
  ++n;
  if (cluster > 1) {
    at[n].id = cudaLaunchAttributeClusterDimension;
    at[n].val.clusterDim.x = cluster; at[n].val.clusterDim.y = 1; at[n].val.clusterDim.z = 1;
    ++n;
  }
  cfg.attrs = at; cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_k1(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  return launch_k(kern, grid, block, smem, st, 1, args...);
}

constexpr int GEMM_MAX_GRID = 160;
constexpr int GEMM_MAX_SPLITS = GEMM_MAX_SLABS_K;
constexpr int QKV_MAX_SLABS = QKV_MAX_SLABS_K;    // pieces per weight tile of the chain's QKV projection (slabs added by the RoPE stage)

// ------------------------------------------------------------------------------------------------ per-device / per-stream state
// Nothing the kernels synchronise through is process-global: the GEMM schedule tables live per DEVICE, the stream-K
// ready flags, the chain kernel's grid barrier and the partial-exchange state per (device, STREAM) - two rings driven on
// two streams never share a flag.  Kernels that wait inside themselves (stream-K owners, the chain's grid barrier) need
// their whole grid resident, so steps enqueued on different streams of one device are ordered behind each other with an
// event (serialise_on): they never run concurrently, whatever the caller's streams allow.
struct SchedKey {
  int split, n_pairs, nkb, max_cl, splits, chunks;
  bool operator<(const SchedKey& o) const { return memcmp(this, &o, sizeof(SchedKey)) < 0; }
};
struct Sched { GemmPiece* dev; int n_cl; int* pair_slabs; int max_slabs; };
struct StreamCtx { int* flags; unsigned long long* bar; };
struct DevCtx {
  int dev = -1, num_sms = 0, max_clusters = 0;       // max_clusters: co-resident 2-CTA clusters of the GEMM / chain kernels
  std::map<SchedKey, Sched> scheds;
  std::map<cudaStream_t, StreamCtx> streams;
  cudaStream_t last_stream = nullptr; bool has_last = false;
  cudaEvent_t last_done = nullptr;
};
static std::mutex g_ctx_mu;
static std::map<int, DevCtx*> g_ctx;

static int get_ctx(DevCtx** out) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  auto it = g_ctx.find(dev);
  if (it != g_ctx.end()) { *out = it->second; return AF_OK; }
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return fail(AF_ERR_UNSUPPORTED, "this library is built for sm_100a only (device %d is sm_%d%d)", dev, prop.major, prop.minor);
  CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(layer_chain_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(layer_chain_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(layer_chain_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(layer_chain_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM_BUDGET));
  CUDA_TRY(cudaFuncSetAttribute(attention_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, att_smem_bytes(128)));
  CUDA_TRY(cudaFuncSetAttribute(attention_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, att_smem_bytes(64)));
  CUDA_TRY(cudaFuncSetAttribute(attention_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, att_smem_bytes(128)));
  CUDA_TRY(cudaFuncSetAttribute(attention_kernel<64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, att_smem_bytes(64)));
  CUDA_TRY(cudaFuncSetAttribute(attention_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, AU_SMEM_BYTES));
  DevCtx* c = new DevCtx();
  c->dev = dev;
  c->num_sms = prop.multiProcessorCount < GEMM_MAX_GRID ? prop.multiProcessorCount : GEMM_MAX_GRID;
  // Stream-K owners and the chain's grid barrier wait for other CTAs of their own grid: size the persistent grids by what
  // the device can hold at once for the actual launch configuration (MPS / green contexts may expose fewer SMs than
  // multiProcessorCount), never by the SM count alone.
  int max_cl = 0;
  {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(2 * GEMM_MAX_GRID); cfg.blockDim = dim3(GEMM_THREADS); cfg.dynamicSmemBytes = GEMM_SMEM_BUDGET;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (cudaOccupancyMaxActiveClusters(&max_cl, layer_chain_kernel<false, false>, &cfg) != cudaSuccess || max_cl < 1) { cudaGetLastError(); max_cl = c->num_sms / 2; }
  }
  c->max_clusters = max_cl < c->num_sms / 2 ? max_cl : c->num_sms / 2;
  if (c->max_clusters < 1) c->max_clusters = 1;
  if (cudaEventCreateWithFlags(&c->last_done, cudaEventDisableTiming) != cudaSuccess) { delete c; return fail(AF_ERR_CUDA, "cudaEventCreate failed"); }
  g_ctx[dev] = c;
  *out = c;
  return AF_OK;
}

static int get_stream_ctx(DevCtx* c, cudaStream_t st, StreamCtx* out) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  auto it = c->streams.find(st);
  if (it != c->streams.end()) { *out = it->second; return AF_OK; }
  StreamCtx sc{};
  uint8_t* mem = nullptr;
  CUDA_TRY(cudaMalloc(&mem, 2048));
  CUDA_TRY(cudaMemset(mem, 0, 2048));
  sc.flags = reinterpret_cast<int*>(mem);                 // [2 * GEMM_MAX_GRID <= 320] ints
  sc.bar = reinterpret_cast<unsigned long long*>(mem + 1536);   // the chain kernel's grid-barrier arrival counter
  c->streams[st] = sc;
  *out = sc;
  return AF_OK;
}

// Order this call's work behind the library work last enqueued on ANOTHER stream of the device (see above).
static int serialise_on(DevCtx* c, cudaStream_t st) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cs);
  if (cs != cudaStreamCaptureStatusNone) return AF_OK;   // a graph being captured orders itself; its replays are the caller's to order
  if (c->has_last && c->last_stream != st) CUDA_TRY(cudaStreamWaitEvent(st, c->last_done, 0));
  return AF_OK;
}
static int serialise_done(DevCtx* c, cudaStream_t st) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cs);
  if (cs == cudaStreamCaptureStatusNone) CUDA_TRY(cudaEventRecord(c->last_done, st));   // (a captured step replays on its own stream)
  c->last_stream = st; c->has_last = true;
  return AF_OK;
}

// debug timeline of the last TRACE_LAUNCHES layer_chain_kernel launches (globaltimer stamps per CTA at every phase end
// and grid-barrier exit), off unless af_debug_trace(1)
constexpr int TRACE_LAUNCHES = 16;
static long long* g_trace = nullptr;
static int g_trace_n = 0;
static bool g_trace_att = false;
struct TraceMeta { int n_phases, grid; };
static TraceMeta g_trace_meta[TRACE_LAUNCHES];
extern "C" int af_debug_trace(int enable) {
  CUDA_TRY(cudaDeviceSynchronize());   // no launch in flight may still hold the buffer
  if (enable && !g_trace) {
    CUDA_TRY(cudaMalloc(&g_trace, sizeof(long long) * TRACE_LAUNCHES * GEMM_MAX_GRID * CH_TRACE_SLOTS));
    CUDA_TRY(cudaMemset(g_trace, 0, sizeof(long long) * TRACE_LAUNCHES * GEMM_MAX_GRID * CH_TRACE_SLOTS));
  }
  if (!enable && g_trace) { cudaFree(g_trace); g_trace = nullptr; }
  g_trace_n = 0;
  g_trace_att = enable == 2;
  return AF_OK;
}
extern "C" int af_debug_trace_read(long long* out, int* meta) {
  if (!g_trace || !out || !meta) return fail(AF_ERR_ARG, "trace is off");
  CUDA_TRY(cudaDeviceSynchronize());
  CUDA_TRY(cudaMemcpy(out, g_trace, sizeof(long long) * TRACE_LAUNCHES * GEMM_MAX_GRID * CH_TRACE_SLOTS, cudaMemcpyDeviceToHost));
  for (int i = 0; i < TRACE_LAUNCHES; ++i) { meta[2 * i] = g_trace_meta[i].n_phases; meta[2 * i + 1] = g_trace_meta[i].grid; }
  return g_trace_n;
}

// threads of the one-block-per-row kernels: two 16-byte accesses per thread and <= 512 threads, so that two blocks fit
// an SM and the ~282 rows of a step run as one wave
static int row_threads_for(int D) { int t = (D / 8 + 31) / 32 * 32; return t < 64 ? 64 : (t > 512 ? 512 : t); }

// split-K pieces per tile of the O / down projections (also the number of slabs the next residual kernel adds)
static int gemm_split_count(const DevCtx* ctx, int n_tiles, int K) {
  const int cluster = n_tiles >= 2 ? 2 : 1;
  const int n_pairs = (n_tiles + cluster - 1) / cluster, nkb = (K + GEMM_BK - 1) / GEMM_BK;
  int s = (cluster == 2 ? ctx->max_clusters : ctx->num_sms) / n_pairs;
  if (s > GEMM_MAX_SPLITS) s = GEMM_MAX_SPLITS;
  if (s > nkb) s = nkb;
  return s < 1 ? 1 : s;
}

// Stream-K ranges: contiguous unit ranges of equal COST, where a range pays its k-blocks plus a charge for every tile
// it touches (the accumulator drain stalls the MMA; a tile entered in its middle is a contributor piece, cheaper than
// an owner / whole tile).  Charges are in k-block units (~0.43 us each at T = 282), from the kernel's timeline.
// Returns the number of ranges used (<= n_max) and fills ub[0..n].
static int streamk_partition(int total, int nkb, int n_max, int* ub) {
  // Ranges shorter than a tile would create pieces in the middle of a tile, which finish last and stall their owner:
  // there the plain uniform split (every tail piece is the first piece of its range) is the better one.
  if (total / n_max < nkb) {
    const int upc = (total + n_max - 1) / n_max, n = (total + upc - 1) / upc;
    for (int i = 0; i <= n; ++i) ub[i] = i * upc < total ? i * upc : total;
    return n;
  }
  const int kTail = 12, kHead = 20;
  auto fill = [&](int cap, int* out) {   // greedy: every range takes as much as `cap` allows; returns ranges used
    int u = 0, n = 0;
    while (u < total) {
      if (n == n_max) return n_max + 1;
      if (out) out[n] = u;
      int cost = 0, e = u;
      while (e < total) {
        const int tile_end = (e / nkb + 1) * nkb;
        const int room = cap - cost - (e % nkb ? kTail : kHead);
        int take = tile_end - e < room ? tile_end - e : room;
        if (take <= 0) { if (e == u) take = 1; else break; }
        cost += (e % nkb ? kTail : kHead) + take;
        e += take;
        if (e < tile_end) break;
      }
      u = e; ++n;
    }
    if (out) out[n] = total;
    return n;
  };
  // smallest cap that fits n_max ranges (one range can always take everything: hi is feasible)
  int lo = total / n_max, hi = total + (total / nkb + 2) * kHead;
  while (lo < hi) { const int mid = (lo + hi) / 2; if (fill(mid, nullptr) <= n_max) hi = mid; else lo = mid + 1; }
  return fill(lo, ub);
}

// ------------------------------------------------------------------------------------------------ GEMM schedules
// Host-built piece lists (GemmPiece, gemm_tcgen05.cuh): which k-blocks of which tile pairs every cluster computes and
// who reduces what.  Built once per (split mode, tile pairs, k-blocks, clusters) and kept on the device.
//   SPLIT_K       one PK_PLAIN piece per cluster: slab `mid` of tile pair c / splits.
//   stream-K      contiguous unit ranges; a range's k-tail piece is its first piece, its k-head piece its last.
//   SPLIT_SLABS   (layer_chain_kernel) contiguous unit ranges of equal length; EVERY piece is a PK_PLAIN piece stored as
//                 slab `mid` = its ordinal inside its tile pair, and the row stage that follows adds a pair's slabs in
//                 that order (pair_slabs[pair] of them, at most `splits`): no CTA waits on another, no fix-up.
// (Two hand-made schedules for the QKV and gate/up shapes - owners with a single piece plus clusters made of
//  contributor pieces only - were built on this table and measured no faster than the ranges; removed.)
constexpr int SPLIT_SLABS = 2;
// SPLIT_K for the FIRST phase of a launch: the CTAs with the highest indices become resident last (on the SMs the previous
// kernel frees last) and have had no time to prefetch weights before griddepcontrol.wait lets the phase start - measured 1.5-2 us
// behind at T = 282, 4 us at T = 6.  So clusters are numbered split-major (the last split of every tile pair sits on the
// last clusters) and the k-ranges shrink linearly from 19/16 of an even share (first split) to 13/16 (last split).
constexpr int SPLIT_K_SKEW = 3;

// Pure host part: the flat [n_cl][GEMM_MAX_PIECES] table (also what af_debug_gemm_schedule returns, for CPU tests).
static int make_schedule(int split, int n_pairs, int nkb, int max_cl, int splits, std::vector<GemmPiece>* flat_out, int* n_cl_out,
                         std::vector<int>* pair_slabs_out = nullptr) {
  if (n_pairs < 1 || nkb < 1 || max_cl < 1 || splits < 1) return fail(AF_ERR_ARG, "bad schedule shape");
  std::vector<std::vector<GemmPiece>> cl;    // pieces per cluster
  auto piece = [](int pair, int kb0, int kb1, int kind, int slot, int n_contrib, int mid) {
    return GemmPiece{pair, kb0, kb1, kind, slot, n_contrib, mid, 0};
  };
  std::vector<int> pair_slabs(n_pairs, 1);
  if (split == SPLIT_K) {
    cl.resize(static_cast<size_t>(n_pairs) * splits);
    for (int c = 0; c < n_pairs * splits; ++c) {
      const int t = c / splits, s = c % splits;
      cl[c].push_back(piece(t, static_cast<int>(1LL * s * nkb / splits), static_cast<int>(1LL * (s + 1) * nkb / splits),
                            PK_PLAIN, 0, 0, s));
    }
    pair_slabs.assign(n_pairs, splits);
  } else if (split == SPLIT_K_SKEW) {
    // split s takes a share of 1 + 3/16 (s = 0) ... 1 - 3/16 (s = splits - 1) of an even one: boundaries from the cumulative shares
    if (nkb < 2 * splits && splits > 1) return fail(AF_ERR_UNSUPPORTED, "GEMM schedule: %d k-blocks cannot feed %d skewed splits", nkb, splits);
    auto kb_at = [&](int sp) {
      if (sp <= 0) return 0;
      if (sp >= splits) return nkb;
      // sum_{i < sp} (16 + 3 - 6 i / (splits - 1)) / (16 splits), in integers
      const long long num = 19LL * sp * (splits - 1) - 3LL * sp * (sp - 1);
      return static_cast<int>((num * nkb + 8LL * splits * (splits - 1)) / (16LL * splits * (splits - 1)));
    };
    cl.resize(static_cast<size_t>(n_pairs) * splits);
    for (int c = 0; c < n_pairs * splits; ++c) {
      const int t = c % n_pairs, sp = c / n_pairs;
      cl[c].push_back(piece(t, kb_at(sp), kb_at(sp + 1), PK_PLAIN, 0, 0, sp));
    }
    pair_slabs.assign(n_pairs, splits);
  } else if (split == SPLIT_SLABS) {
    // Ranges of equal COST over all clusters: a range pays its k-blocks plus kSlabCharge k-blocks for every tile pair it
    // touches (each piece ends in an accumulator drain and a pipeline refill, ~9 k-blocks' worth at T = 282; with equal LENGTHS the two
    // thirds of the clusters whose range crosses a pair boundary finished 3 us after the others).  Never shorter than
    // lmin, so that a tile pair is cut into at most `splits` pieces.
    const int total = n_pairs * nkb;
    constexpr int kSlabCharge = 9;
    int lmin = 1;
    if (splits > 1) lmin = (nkb - 1 + splits - 2) / (splits - 1);
    else lmin = nkb;
    if (lmin < 1) lmin = 1;
    std::vector<int> ub;   // range c = [ub[c], ub[c + 1])
    auto cut = [&](long long cap, std::vector<int>* out) {   // greedy: every range as long as `cap` allows
      out->assign(1, 0);
      int a = 0;
      while (a < total) {
        int b = a + lmin < total ? a + lmin : total;
        if (splits == 1) { b = (b + nkb - 1) / nkb * nkb; if (b > total) b = total; }
        auto cost = [&](int e) { return static_cast<long long>(e - a) + kSlabCharge * ((e - 1) / nkb - a / nkb + 1); };
        while (b < total) {
          const int nb = splits == 1 ? (b + nkb < total ? b + nkb : total) : b + 1;
          if (cost(nb) > cap) break;
          b = nb;
        }
        out->push_back(b);
        a = b;
      }
      return static_cast<int>(out->size()) - 1;
    };
    long long lo = 1, hi = static_cast<long long>(total) + kSlabCharge * (n_pairs + 1);
    while (lo < hi) {   // the smallest cap that fits max_cl ranges
      const long long mid_cap = (lo + hi) / 2;
      std::vector<int> tmp;
      if (cut(mid_cap, &tmp) <= max_cl) hi = mid_cap; else lo = mid_cap + 1;
    }
    const int n = cut(lo, &ub);
    if (n > max_cl) return fail(AF_ERR_UNSUPPORTED, "GEMM schedule: %d ranges for %d clusters", n, max_cl);
    cl.resize(n);
    pair_slabs.assign(n_pairs, 0);
    for (int c = 0; c < n; ++c) {
      int u = ub[c];
      const int end = ub[c + 1];
      while (u < end) {
        const int t = u / nkb, kb0 = u - t * nkb;
        const int kb1 = end - t * nkb < nkb ? end - t * nkb : nkb;
        cl[c].push_back(piece(t, kb0, kb1, PK_PLAIN, 0, 0, pair_slabs[t]++));
        u = t * nkb + kb1;
      }
    }
    for (int t = 0; t < n_pairs; ++t)
      if (pair_slabs[t] > splits) return fail(AF_ERR_UNSUPPORTED, "GEMM schedule: %d slabs of one tile pair (max %d)", pair_slabs[t], splits);
  } else {
    // stream-K ranges (cost-balanced when a range is longer than a tile)
    const int total = n_pairs * nkb;
    std::vector<int> ub(max_cl + 2);
    const int n = streamk_partition(total, nkb, total < max_cl ? total : max_cl, ub.data());
    cl.resize(n);
    for (int c = 0; c < n; ++c) {
      int u = ub[c];
      while (u < ub[c + 1]) {
        const int t = u / nkb, kb0 = u - t * nkb;
        const int kb1 = ub[c + 1] - t * nkb < nkb ? ub[c + 1] - t * nkb : nkb;
        if (kb0 > 0) {
          cl[c].push_back(piece(t, kb0, kb1, PK_CONTRIB, c, 0, 0));          // slot = its cluster (one tail per range)
        } else if (kb1 < nkb) {
          int nc = 0;
          while (c + 1 + nc < n && ub[c + 1 + nc] < (t + 1) * nkb) ++nc;     // ranges that start inside this tile
          cl[c].push_back(piece(t, 0, kb1, PK_OWNER, c + 1, nc, 0));
        } else {
          cl[c].push_back(piece(t, 0, nkb, PK_PLAIN, 0, 0, 0));
        }
        u = t * nkb + kb1;
      }
    }
  }
  const int n_cl = static_cast<int>(cl.size());
  std::vector<GemmPiece>& flat = *flat_out;
  flat.assign(static_cast<size_t>(n_cl) * GEMM_MAX_PIECES, GemmPiece{-1, 0, 0, 0, 0, 0, 0, 0});
  for (int c = 0; c < n_cl; ++c) {
    if (static_cast<int>(cl[c].size()) > GEMM_MAX_PIECES - 1)
      return fail(AF_ERR_UNSUPPORTED, "GEMM schedule: %zu pieces in one cluster (max %d)", cl[c].size(), GEMM_MAX_PIECES - 1);
    for (size_t i = 0; i < cl[c].size(); ++i) flat[static_cast<size_t>(c) * GEMM_MAX_PIECES + i] = cl[c][i];
  }
  *n_cl_out = n_cl;
  if (pair_slabs_out) *pair_slabs_out = pair_slabs;
  return AF_OK;
}

// The device copy has at least max_cl rows (clusters beyond n_cl find an empty list), so that kernels whose grid is the
// whole device (layer_chain_kernel) can index it with any cluster id.
// chunks = 2 (the chain with 512 < T <= 1024): every piece appears twice, for token chunk 0 and 1 (GemmPiece::pad), adjacent in
// its cluster's list - the second pass re-reads the same weight k-range while it is still in L2.
static int build_schedule(DevCtx* ctx, int split, int n_pairs, int nkb, int max_cl, int splits, Sched* out, int chunks = 1) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  const SchedKey key{split, n_pairs, nkb, max_cl, splits, chunks};
  auto it = ctx->scheds.find(key);
  if (it != ctx->scheds.end()) { *out = it->second; return AF_OK; }
  std::vector<GemmPiece> flat;
  std::vector<int> pair_slabs;
  int n_cl = 0;
  const int rc = make_schedule(split, n_pairs, nkb, max_cl, splits, &flat, &n_cl, &pair_slabs);
  if (rc) return rc;
  if (chunks == 2) {
    std::vector<GemmPiece> two(flat.size(), GemmPiece{-1, 0, 0, 0, 0, 0, 0, 0});
    for (int c = 0; c < n_cl; ++c) {
      int n = 0;
      for (int i = 0; i < GEMM_MAX_PIECES && flat[static_cast<size_t>(c) * GEMM_MAX_PIECES + i].pair >= 0; ++i) {
        if (n + 2 > GEMM_MAX_PIECES - 1) return fail(AF_ERR_UNSUPPORTED, "GEMM schedule: too many pieces in one cluster for two token chunks");
        for (int ch = 0; ch < 2; ++ch) {
          GemmPiece q = flat[static_cast<size_t>(c) * GEMM_MAX_PIECES + i];
          q.pad = ch;
          two[static_cast<size_t>(c) * GEMM_MAX_PIECES + n++] = q;
        }
      }
    }
    flat.swap(two);
  }
  if (n_cl < max_cl) flat.resize(static_cast<size_t>(max_cl) * GEMM_MAX_PIECES, GemmPiece{-1, 0, 0, 0, 0, 0, 0, 0});
  Sched sc{nullptr, n_cl, nullptr, 0};
  for (int v : pair_slabs) sc.max_slabs = v > sc.max_slabs ? v : sc.max_slabs;
  CUDA_TRY(cudaMalloc(&sc.dev, flat.size() * sizeof(GemmPiece)));
  CUDA_TRY(cudaMemcpy(sc.dev, flat.data(), flat.size() * sizeof(GemmPiece), cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMalloc(&sc.pair_slabs, pair_slabs.size() * sizeof(int)));
  CUDA_TRY(cudaMemcpy(sc.pair_slabs, pair_slabs.data(), pair_slabs.size() * sizeof(int), cudaMemcpyHostToDevice));
  ctx->scheds[key] = sc;
  *out = sc;
  return AF_OK;
}

static size_t gemm_partial_bytes() { return static_cast<size_t>(GEMM_MAX_GRID) * GEMM_MAX_TOK * GEMM_BM * sizeof(float); }

// One projection over all T packed rows (token chunks of <= 512 rows per launch).  `proto` carries the weight
// layout (n_parts / part_rows / a_pair), the split mode and the epilogue fields; the decomposition is filled here.
static int launch_gemm(int cat, cudaStream_t st, GemmParams proto, const OutView& ov, /* proto.w_fp16 set by the caller */ const void* x, int x_rows_cap,
                       const void* const* w, int T) {
  DevCtx* ctx = nullptr;
  int rc = get_ctx(&ctx);
  if (rc) return rc;
  if (T <= 0) return AF_OK;
  StreamCtx sctx;
  if ((rc = get_stream_ctx(ctx, st, &sctx))) return rc;
  const int n_chunks = (T + GEMM_MAX_TOK - 1) / GEMM_MAX_TOK;
  const int chunk = (T + n_chunks - 1) / n_chunks;
  for (int tok0 = 0; tok0 < T; tok0 += chunk) {
    const int Tc = (T - tok0 < chunk) ? (T - tok0) : chunk;
    GemmParams p = proto;
    int n_pad = (Tc + 15) / 16 * 16;
    if (n_pad <= 256) { p.n1 = n_pad; p.n2 = 0; }
    else { p.n1 = ((Tc + 1) / 2 + 15) / 16 * 16; p.n2 = p.n1; n_pad = 2 * p.n1; }
    const int box_rows = p.a_pair == 1 ? 16 : GEMM_BM;
    const int n_tiles = p.a_pair ? (p.part_rows + 63) / 64 : p.n_parts * ((p.part_rows + GEMM_BM - 1) / GEMM_BM);
    p.tiles_per_part = (p.part_rows + GEMM_BM - 1) / GEMM_BM;
    p.num_kb = (p.K + GEMM_BK - 1) / GEMM_BK; p.T = Tc; p.tok0 = tok0;
    p.xh = p.n2 > 0 ? p.n1 : p.n1 / 2;
    p.n_tiles = n_tiles;
    p.cluster = n_tiles >= 2 ? 2 : 1;
    const int n_pairs = (n_tiles + p.cluster - 1) / p.cluster;     // work units are (tile pair, k-block) per cluster
    const int max_cl = p.cluster == 2 ? ctx->max_clusters : ctx->num_sms;
    p.splits = p.split == SPLIT_K ? gemm_split_count(ctx, n_tiles, p.K) : 1;
    Sched sc;
    if ((rc = build_schedule(ctx, p.split, n_pairs, p.num_kb, max_cl, p.splits, &sc))) return rc;
    p.sched = sc.dev;
    p.n_cl = sc.n_cl;
    const int grid = sc.n_cl * p.cluster;
    p.mma2 = (p.cluster == 2 && p.w_fp16) ? 1 : 0;
    const int stage_bytes = GEMM_BM * GEMM_BK * 2 + (p.mma2 ? n_pad / 2 : n_pad) * GEMM_BK * 2;
    // epilogue staging: two 4 KB buffers per warp, or one 2 KB buffer when that buys a pipeline stage (the main loop
    // is bound by TMA latency x stages in flight)
    // candidates, largest staging first; a smaller one is taken when it buys a pipeline stage (the main loop needs
    // ~160 KB of loads in flight), down to one 2 KB buffer per warp
    const int cand[3][2] = {{4096, 2}, {2048, 2}, {2048, 1}};
    if (ov.elem_bytes == 2) return fail(AF_ERR_UNSUPPORTED, "GEMM outputs are fp16 or fp32");
    p.out_f16 = ov.elem_bytes == -2 ? 2 : 0;
    p.part_f16 = p.out_f16 ? 1 : 0;   // fp16 outputs take fp16 partials (both in the fragment layout), fp32 take fp32
    if (p.out_f16) {
      if (ov.features % 8 || ov.ld_tok % 8 || ov.ld_mid % 8 || (reinterpret_cast<uintptr_t>(ov.ptr) & 15))
        return fail(AF_ERR_ARG, "fp16 GEMM output needs 16-byte aligned rows (features %d, ld %lld/%lld)", ov.features, ov.ld_tok, ov.ld_mid);
      p.out = ov.ptr; p.out_ld_tok = ov.ld_tok; p.out_ld_mid = ov.ld_mid; p.out_features = ov.features;
    }
    int stages = 0;
    // (fp16 outputs: one 2 KB image per warp, read back by the warp itself - nothing asynchronous to wait for)
    for (int i = p.out_f16 ? 2 : 0; i < 3; ++i) {
      const int st_i = (GEMM_SMEM_BUDGET - 1024 - GEMM_EPI_WARPS * cand[i][0] * cand[i][1]) / stage_bytes;
      if (st_i > stages && (stages < kMinStages || stages == 0)) { stages = st_i; p.stg_bytes = cand[i][0]; p.stg_bufs = cand[i][1]; }
    }
    const int xch_bytes = GEMM_EPI_WARPS * p.stg_bytes * p.stg_bufs;
    if (stages > GEMM_MAX_STAGES) stages = GEMM_MAX_STAGES;
    if (stages < 2) return fail(AF_ERR_UNSUPPORTED, "GEMM stage does not fit shared memory");
    p.stages = stages; p.flags = sctx.flags;
    p.w_pre = kWeightStagesBeforeWait < stages ? kWeightStagesBeforeWait : stages;
    CUtensorMap mw[3], mx;
    for (int i = 0; i < 3; ++i) {
      const int n_w = p.a_pair == 1 ? 2 : (p.a_pair == 2 ? 1 : p.n_parts);
      rc = get_map(w[i < n_w ? i : 0], p.a_pair == 2 ? n_tiles * GEMM_BM : p.part_rows, p.K, box_rows, &mw[i]);
      if (rc) return rc;
    }
    rc = get_map(x, x_rows_cap, p.K, p.mma2 ? p.n1 / 2 : p.xh, &mx);
    if (rc) return rc;
    CUtensorMap mo, mp;
    if ((rc = get_out_map(ov, p.stg_bytes, &mo))) return rc;
    if (p.part_f16) {
      mp = mo;   // fp16 partials are raw 2 KB staging images [slot][32-token chunk][quadrant], written by 1-D bulk copies
    } else {     // fp32 stream-K partials [slot][512 tokens][128 features], box = 32 features x 32 (or 16) tokens of one slot
      const unsigned long long dims[3] = {GEMM_BM, GEMM_MAX_TOK, GEMM_MAX_GRID};
      const unsigned long long strides[2] = {GEMM_BM * 4ull, GEMM_BM * 4ull * GEMM_MAX_TOK};
      const unsigned box[3] = {32u, p.stg_bytes < 4096 ? 16u : 32u, 1u};
      if ((rc = get_map_nd(p.partial, 4, 3, dims, strides, box, 0, &mp))) return rc;
    }
    const size_t smem = static_cast<size_t>(stages) * stage_bytes + xch_bytes + 1024;
    {
      ProfScope ps(cat, st);
      auto kern = p.mma2 ? (p.out_f16 ? gemm_tcgen05_kernel<true, true> : gemm_tcgen05_kernel<true, false>)
                         : (p.out_f16 ? gemm_tcgen05_kernel<false, true> : gemm_tcgen05_kernel<false, false>);
      cudaError_t e = launch_k(kern, dim3(grid), dim3(GEMM_THREADS), smem, st, p.cluster, mw[0], mw[1], mw[2], mx, mo, mp, p);
      if (e != cudaSuccess) return fail(AF_ERR_CUDA, "launch of gemm_tcgen05_kernel failed: %s", cudaGetErrorString(e));
    }
    rc = check_launch("gemm_tcgen05_kernel");
    if (rc) return rc;
  }
  return AF_OK;
}

// ------------------------------------------------------------------------------------------------ layer chain (chain.cuh)
// Host side of layer_chain_kernel: phases are appended to a ChainArgs (tensor maps deduplicated), then one launch.
struct ChainBuilder {
  ChainArgs a;
  int n_maps = 0;
  DevCtx* ctx = nullptr;
  int max_rows = 0;          // row capacity of the workspace buffers the activation maps cover
  bool fp8 = false;          // AF_WEIGHTS_FP8: weight matrices are E4M3 codes + per-output-channel scales
  int chunks = 1;            // 2: 512 < T <= 1024, every piece once per token chunk
  ChainBuilder() { memset(&a, 0, sizeof a); }
  int add_map(const CUtensorMap& m) {
    for (int i = 0; i < n_maps; ++i)
      if (memcmp(&a.maps[i], &m, sizeof m) == 0) return i;
    if (n_maps == CH_MAX_MAPS) return -1;
    a.maps[n_maps] = m;
    return n_maps++;
  }
  ChainPhase* next() { return a.n_phases < CH_MAX_PHASES ? &a.ph[a.n_phases++] : nullptr; }
};

// One projection phase: y = x W^T over n_parts weight matrices stacked along the feature axis (a_pair = 2: gate | up
// interleaved by af_prepare_gate_up).  split: SPLIT_K / SPLIT_SLABS (EPI_STORE, slabs) or SPLIT_STREAMK (EPI_SWIGLU).
static int chain_add_gemm(ChainBuilder& b, const void* const* w, const float* const* scales, int n_parts, int part_rows, int a_pair, int K,
                          int split, int max_slabs, int epi, const void* x, act_t* out, long long out_ld_tok, long long out_ld_slab,
                          int out_features, const int** pair_slabs_out, int* n_slabs_out) {
  ChainPhase* P = b.next();
  if (!P) return fail(AF_ERR_UNSUPPORTED, "chain: too many phases");
  P->kind = CH_GEMM;
  const int n_tiles = a_pair ? (part_rows + 63) / 64 : n_parts * ((part_rows + GEMM_BM - 1) / GEMM_BM);
  P->part_rows = part_rows; P->tiles_per_part = (part_rows + GEMM_BM - 1) / GEMM_BM; P->a_pair = a_pair;
  P->n_tiles = n_tiles; P->num_kb = (K + GEMM_BK - 1) / GEMM_BK; P->epi = epi;
  const int n_pairs = (n_tiles + 1) / 2;
  int splits = max_slabs;
  if (split == SPLIT_K) {
    splits = gemm_split_count(b.ctx, n_tiles, K);
    if (P == &b.a.ph[0] && splits > 1 && P->num_kb >= 4 * splits) split = SPLIT_K_SKEW;   // the launch's first phase: late-resident clusters get the short pieces
  }
  Sched sc;
  int rc = build_schedule(b.ctx, split, n_pairs, P->num_kb, b.ctx->max_clusters, split == SPLIT_STREAMK ? 1 : splits, &sc, b.chunks);
  if (rc) return rc;
  P->sched = sc.dev;
  if (pair_slabs_out) *pair_slabs_out = sc.pair_slabs;
  if (n_slabs_out) *n_slabs_out = sc.max_slabs;
  for (int i = 0; i < 3; ++i) {
    CUtensorMap m;
    const int n_w = a_pair ? 1 : n_parts;
    const int w_rows = a_pair ? n_tiles * GEMM_BM : part_rows;
    if ((rc = b.fp8 ? get_map_fp8(w[i < n_w ? i : 0], w_rows, K, &m) : get_map(w[i < n_w ? i : 0], w_rows, K, GEMM_BM, &m))) return rc;
    if ((P->w_map[i] = b.add_map(m)) < 0) return fail(AF_ERR_UNSUPPORTED, "chain: too many tensor maps");
    P->scale[i] = (b.fp8 && scales) ? scales[i < (a_pair ? 2 : n_parts) ? i : 0] : nullptr;
    if (b.fp8 && !P->scale[i]) return fail(AF_ERR_ARG, "AF_WEIGHTS_FP8 needs af_weights.scales");
  }
  CUtensorMap mx;
  if ((rc = get_map(x, b.max_rows, K, b.a.n1 / 2, &mx))) return rc;
  if ((P->x_map = b.add_map(mx)) < 0) return fail(AF_ERR_UNSUPPORTED, "chain: too many tensor maps");
  if (out_features % 8 || out_ld_tok % 8 || out_ld_slab % 8 || (reinterpret_cast<uintptr_t>(out) & 15))
    return fail(AF_ERR_ARG, "chain: fp16 GEMM output needs 16-byte aligned rows");
  P->out = out; P->out_ld_tok = out_ld_tok; P->out_ld_slab = out_ld_slab; P->out_features = out_features;
  return AF_OK;
}

static int chain_add_rows(ChainBuilder& b, const void* src, int embed, int n_slabs, long long slab_stride, const void* gain, act_t* xn) {
  ChainPhase* P = b.next();
  if (!P) return fail(AF_ERR_UNSUPPORTED, "chain: too many phases");
  P->kind = CH_ROWS; P->src = src; P->embed = embed; P->n_slabs = n_slabs; P->slab_stride = slab_stride;
  P->gain = reinterpret_cast<const __nv_bfloat16*>(gain); P->xn = xn;
  return AF_OK;
}

static int chain_add_rope(ChainBuilder& b, const act_t* qkv_slabs, long long slab_stride, const int* pair_slabs, act_t* q_out, act_t* kv_layer) {
  ChainPhase* P = b.next();
  if (!P) return fail(AF_ERR_UNSUPPORTED, "chain: too many phases");
  P->kind = CH_ROPE; P->src = qkv_slabs; P->slab_stride = slab_stride; P->pair_slabs = pair_slabs; P->q_out = q_out; P->kv_layer = kv_layer;
  return AF_OK;
}

static int chain_add_attn(ChainBuilder& b, const AuArgs& att) {   // must be the launch's last phase
  if (b.a.n_phases >= CH_MAX_PHASES) return fail(AF_ERR_UNSUPPORTED, "chain: too many phases");
  ChainPhase& P = b.a.ph[b.a.n_phases++];
  P = ChainPhase{};
  P.kind = CH_ATTN;
  b.a.att = att;
  b.a.att_on = 1;
  return AF_OK;
}

static int chain_launch(ChainBuilder& b, cudaStream_t st, int cat) {
  const int n_pad = b.a.n1 + b.a.n2;
  const int stage_bytes = GEMM_BM * GEMM_BK * 2 + (n_pad / 2) * GEMM_BK * 2;   // (FP8: the raw tile lands inside the fp16 tile's slot)
  int stages = (GEMM_SMEM_BUDGET - 1024 - GEMM_EPI_WARPS * 2048) / stage_bytes;
  if (stages > GEMM_MAX_STAGES) stages = GEMM_MAX_STAGES;
  if (stages < 2) return fail(AF_ERR_UNSUPPORTED, "chain: a stage does not fit shared memory");
  b.a.stages = stages;
  const int grid = 2 * b.ctx->max_clusters;
  b.a.trace = nullptr;
  if (g_trace && !g_trace_att && grid <= GEMM_MAX_GRID) {
    b.a.trace = g_trace + static_cast<size_t>(g_trace_n % TRACE_LAUNCHES) * GEMM_MAX_GRID * CH_TRACE_SLOTS;
    g_trace_meta[g_trace_n % TRACE_LAUNCHES] = {b.a.n_phases, grid};
    ++g_trace_n;
  }
  size_t smem = static_cast<size_t>(stages) * stage_bytes + GEMM_EPI_WARPS * 2048 + 1024;
  if (b.a.att_on) {   // the attention units' tiles and state reuse the stage ring
    if (b.a.ph[b.a.n_phases - 1].kind != CH_ATTN) return fail(AF_ERR_UNSUPPORTED, "chain: attention must be the last phase");
    const size_t need = static_cast<size_t>(AU_TILE_BYTES) + sizeof(AuAux) + 1024;
    if (need > static_cast<size_t>(GEMM_SMEM_BUDGET)) return fail(AF_ERR_UNSUPPORTED, "chain: attention tiles do not fit shared memory");
    if (smem < need) smem = need;
  }
  cudaError_t e;
  { ProfScope ps(cat, st); e = launch_k(b.chunks == 2 ? (b.fp8 ? layer_chain_kernel<true, true> : layer_chain_kernel<false, true>)
                                                         : (b.fp8 ? layer_chain_kernel<true, false> : layer_chain_kernel<false, false>), dim3(grid), dim3(GEMM_THREADS), smem, st, 2, b.a); }
  if (e != cudaSuccess) return fail(AF_ERR_CUDA, "launch of layer_chain_kernel failed: %s", cudaGetErrorString(e));
  return check_launch("layer_chain_kernel");
}

// ------------------------------------------------------------------------------------------------ ring handle
struct af_ring {
  af_model_cfg cfg;
  af_ring_cfg rc;
  act_t* kv;                    // caller-owned, fp16
  std::vector<int> base, len;   // host mirror, authoritative for validation (a0, a9)
  int* tables = nullptr;        // library-owned device ints backing StepTables
  StepTables tb{};
  int* n_items_dev = nullptr;
  int* att_sched = nullptr;
  float2* rope_tab = nullptr;   // [C][hd/2]
  int max_rows = 0;
  int last_T = 0;
  int window = 0;               // f3: 0 = none (start_pos + len <= C), else rows see the last `window` positions
  int max_pos = 0;              // positions stay below this (rows of the RoPE table); = C without a window
};

static int check_cfg(const af_model_cfg* c) {
  if (!c) return fail(AF_ERR_ARG, "null model cfg");
  if (c->d_model <= 0 || c->n_layers <= 0 || c->n_heads <= 0 || c->ffn <= 0 || c->vocab <= 0)
    return fail(AF_ERR_ARG, "non-positive model dimension");
  if (c->head_dim != 64 && c->head_dim != 128) return fail(AF_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", c->head_dim);
  if (c->d_model != c->n_heads * c->head_dim) return fail(AF_ERR_UNSUPPORTED, "d_model != n_heads*head_dim");
  if (c->d_model % 8 || c->ffn % 8) return fail(AF_ERR_UNSUPPORTED, "d_model and ffn must be multiples of 8");
  return AF_OK;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

extern "C" size_t af_ring_bytes(const af_model_cfg* c, const af_ring_cfg* r) {
  if (!c || !r) return 0;
  return static_cast<size_t>(2) * c->n_layers * r->n_regions * c->n_heads * r->capacity * c->head_dim * 2;
}

// workspace = fixed part (stream-K partials) + per-row part; the carve depends only on (pointer, bytes)
static size_t ws_per_row(const af_model_cfg* c) {
  const size_t D = c->d_model, F = c->ffn;
  // xn, qkv (QKV_MAX_SLABS slabs), q_rot, attn, h (fp16) + split-K slabs of the O / down projections
  return align_up((D + QKV_MAX_SLABS * 3 * D + D + D + F) * 2 + GEMM_MAX_SPLITS * D * 4, 256);
}
static size_t ws_fixed() { return align_up(gemm_partial_bytes(), 256) + 8 * 256; }

extern "C" size_t af_workspace_bytes(const af_model_cfg* c, int32_t max_rows, int32_t max_segs) {
  (void)max_segs;
  if (!c || max_rows < 0) return 0;
  const size_t rows = align_up(static_cast<size_t>(max_rows < 16 ? 16 : max_rows), 16);
  return ws_fixed() + rows * ws_per_row(c);
}

struct Workspace {
  float* partial;        // stream-K partials [grid][n_pad][128]
  float* split;          // split-K slabs [GEMM_MAX_SPLITS][max_rows][D]
  act_t *xn, *qkv, *q_rot, *attn, *h;   // fp16 activations (qkv: QKV_MAX_SLABS slabs of [max_rows][3D]; the per-stage path uses the first)
  int max_rows;
};
static int carve(const af_model_cfg* c, void* ws, size_t bytes, int need_rows, Workspace* o) {
  if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255)) return fail(AF_ERR_ARG, "workspace must be 256-byte aligned");
  if (bytes < ws_fixed() + 16 * ws_per_row(c)) return fail(AF_ERR_WORKSPACE, "workspace of %zu bytes is too small", bytes);
  size_t rows = (bytes - ws_fixed()) / ws_per_row(c);
  rows = rows / 16 * 16;
  if (rows > 65536) rows = 65536;
  if (static_cast<size_t>(need_rows) > rows)
    return fail(AF_ERR_WORKSPACE, "workspace holds %zu rows, %d needed (use af_workspace_bytes)", rows, need_rows);
  uint8_t* p = reinterpret_cast<uint8_t*>(ws);
  const size_t D = c->d_model, F = c->ffn;
  auto take = [&](size_t n) { uint8_t* q = p; p += align_up(n, 256); return q; };
  o->partial = reinterpret_cast<float*>(take(gemm_partial_bytes()));
  o->split = reinterpret_cast<float*>(take(GEMM_MAX_SPLITS * rows * D * 4));
  o->xn = reinterpret_cast<act_t*>(take(rows * D * 2));
  o->qkv = reinterpret_cast<act_t*>(take(QKV_MAX_SLABS * rows * 3 * D * 2));
  o->q_rot = reinterpret_cast<act_t*>(take(rows * D * 2));
  o->attn = reinterpret_cast<act_t*>(take(rows * D * 2));
  o->h = reinterpret_cast<act_t*>(take(rows * F * 2));
  o->max_rows = static_cast<int>(rows);
  return AF_OK;
}

extern "C" int af_ring_create(const af_model_cfg* c, const af_ring_cfg* r, void* kv_mem, size_t kv_bytes, af_ring** out) {
  int rc = check_cfg(c);
  if (rc) return rc;
  if (!r || !out || !kv_mem) return fail(AF_ERR_ARG, "null argument");
  if (r->n_regions <= 0 || r->capacity <= 0) return fail(AF_ERR_ARG, "ring needs n_regions > 0 and capacity > 0");
  if (reinterpret_cast<uintptr_t>(kv_mem) & 255) return fail(AF_ERR_ARG, "kv_mem must be 256-byte aligned");
  if (kv_bytes < af_ring_bytes(c, r)) return fail(AF_ERR_WORKSPACE, "kv_mem of %zu bytes < af_ring_bytes %zu", kv_bytes, af_ring_bytes(c, r));
  DevCtx* ctx = nullptr;
  if ((rc = get_ctx(&ctx))) return rc;
  af_ring* g = new af_ring();
  g->cfg = *c; g->rc = *r; g->kv = reinterpret_cast<act_t*>(kv_mem);
  g->base.assign(r->n_regions, 0); g->len.assign(r->n_regions, 0);
  g->max_pos = r->capacity;
  const long long cap_rows = static_cast<long long>(r->n_regions) * r->capacity;
  g->max_rows = static_cast<int>(cap_rows > 65536 ? 65536 : cap_rows);
  const size_t n_int = 5 * AF_MAX_SEGS + 3 * static_cast<size_t>(g->max_rows) + 4 * (g->max_rows / ATT_BQ + AF_MAX_SEGS) + 1 + 2;
  cudaError_t e = cudaMalloc(&g->tables, n_int * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&g->rope_tab, static_cast<size_t>(r->capacity) * (c->head_dim / 2) * sizeof(float2));
  if (e != cudaSuccess) { cudaFree(g->tables); delete g; return fail(AF_ERR_CUDA, "cudaMalloc: %s", cudaGetErrorString(e)); }
  int* p = g->tables;
  g->tb.seg_req = p; p += AF_MAX_SEGS; g->tb.seg_start = p; p += AF_MAX_SEGS; g->tb.seg_len = p; p += AF_MAX_SEGS;
  g->tb.seg_row0 = p; p += AF_MAX_SEGS; g->tb.seg_base = p; p += AF_MAX_SEGS;
  g->tb.row_req = p; p += g->max_rows; g->tb.row_pos = p; p += g->max_rows; g->tb.row_slot = p; p += g->max_rows;
  const int max_items = g->max_rows / ATT_BQ + AF_MAX_SEGS;
  g->tb.item_seg = p; p += max_items; g->tb.item_q0 = p; p += max_items; g->tb.item_tmp = p; p += 2 * max_items;
  g->n_items_dev = p; ++p;
  g->att_sched = p;   // attention_umma_kernel's unit counters: zero between launches
  if (cudaMemset(g->att_sched, 0, 2 * sizeof(int)) != cudaSuccess) { cudaFree(g->tables); cudaFree(g->rope_tab); delete g; return fail(AF_ERR_CUDA, "cudaMemset failed"); }
  const int n = r->capacity * (c->head_dim / 2);
  rope_table_kernel<<<(n + 255) / 256, 256>>>(g->rope_tab, r->capacity, c->head_dim, static_cast<double>(c->rope_theta));
  rc = check_launch("rope_table_kernel");
  if (rc == AF_OK && cudaDeviceSynchronize() != cudaSuccess) rc = fail(AF_ERR_CUDA, "rope table build failed");
  if (rc) { cudaFree(g->tables); cudaFree(g->rope_tab); delete g; return rc; }
  *out = g;
  return AF_OK;
}

extern "C" int af_ring_destroy(af_ring* g) {
  if (!g) return AF_OK;
  cudaFree(g->tables);
  cudaFree(g->rope_tab);
  delete g;
  return AF_OK;
}

extern "C" int af_ring_reset_slot(af_ring* g, int32_t req, int32_t new_base) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  if (req < 0 || req >= g->rc.n_regions) return fail(AF_ERR_SEGMENT, "req_id %d outside [0,%d)", req, g->rc.n_regions);
  const int C = g->rc.capacity;
  g->base[req] = new_base >= 0 ? new_base % C : (g->base[req] + g->len[req]) % C;
  g->len[req] = 0;
  return AF_OK;
}

extern "C" int af_ring_set_window(af_ring* g, int32_t window, int32_t max_pos) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  const int C = g->rc.capacity;
  if (window < 0 || window > C) return fail(AF_ERR_ARG, "window %d outside [0, capacity %d]", window, C);
  if (window == 0) max_pos = C;
  if (max_pos < C) return fail(AF_ERR_ARG, "max_pos %d < capacity %d", max_pos, C);
  for (int r = 0; r < g->rc.n_regions; ++r)
    if (g->len[r] != 0) return fail(AF_ERR_POSITION, "af_ring_set_window needs every region empty (request %d has %d tokens)", r, g->len[r]);
  if (max_pos != g->max_pos) {   // the RoPE table has one row per position
    float2* tab = nullptr;
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMalloc(&tab, static_cast<size_t>(max_pos) * (g->cfg.head_dim / 2) * sizeof(float2)));
    const int n = max_pos * (g->cfg.head_dim / 2);
    rope_table_kernel<<<(n + 255) / 256, 256>>>(tab, max_pos, g->cfg.head_dim, static_cast<double>(g->cfg.rope_theta));
    int rc = check_launch("rope_table_kernel");
    if (rc == AF_OK && cudaDeviceSynchronize() != cudaSuccess) rc = fail(AF_ERR_CUDA, "rope table build failed");
    if (rc) { cudaFree(tab); return rc; }
    cudaFree(g->rope_tab);
    g->rope_tab = tab;
  }
  g->window = window; g->max_pos = max_pos;
  return AF_OK;
}

extern "C" int af_ring_get_state(const af_ring* g, int32_t req, int32_t* base, int32_t* len) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  if (req < 0 || req >= g->rc.n_regions) return fail(AF_ERR_SEGMENT, "req_id %d outside [0,%d)", req, g->rc.n_regions);
  if (base) *base = g->base[req];
  if (len) *len = g->len[req];
  return AF_OK;
}

extern "C" int af_debug_set_len(af_ring* g, int32_t req, int32_t len) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  if (req < 0 || req >= g->rc.n_regions) return fail(AF_ERR_SEGMENT, "req_id %d outside [0,%d)", req, g->rc.n_regions);
  if (len < 0 || len > g->max_pos) return fail(AF_ERR_CAPACITY, "len %d outside [0,%d]", len, g->max_pos);
  g->len[req] = len;
  return AF_OK;
}

extern "C" int af_debug_row_map(const af_ring* g, int32_t* row_req, int32_t* row_pos, int32_t* row_slot, int32_t n) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  if (n < 0 || n > g->last_T) return fail(AF_ERR_ARG, "n = %d but the last step had %d rows", n, g->last_T);
  CUDA_TRY(cudaDeviceSynchronize());
  if (row_req) CUDA_TRY(cudaMemcpy(row_req, g->tb.row_req, n * sizeof(int), cudaMemcpyDeviceToHost));
  if (row_pos) CUDA_TRY(cudaMemcpy(row_pos, g->tb.row_pos, n * sizeof(int), cudaMemcpyDeviceToHost));
  if (row_slot) CUDA_TRY(cudaMemcpy(row_slot, g->tb.row_slot, n * sizeof(int), cudaMemcpyDeviceToHost));
  return AF_OK;
}

extern "C" int af_convert_bf16_to_fp16(const void* src, void* dst, size_t n, void* cuda_stream) {
  if (!src || !dst || (n % 8)) return fail(AF_ERR_ARG, "null pointer or n_elems not a multiple of 8");
  if ((reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst)) & 15) return fail(AF_ERR_ARG, "pointers must be 16-byte aligned");
  if (n == 0) return AF_OK;
  const size_t n_vec = n / 8;
  convert_bf16_to_fp16_kernel<<<static_cast<unsigned>((n_vec + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(
      reinterpret_cast<const uint4*>(src), reinterpret_cast<uint4*>(dst), n_vec);
  return check_launch("convert_bf16_to_fp16_kernel");
}

extern "C" int af_argmax_rows(const float* logits, int32_t n_rows, int32_t vocab, int32_t* tokens_out, void* cuda_stream) {
  if (n_rows < 0 || vocab <= 0 || (n_rows > 0 && (!logits || !tokens_out))) return fail(AF_ERR_ARG, "af_argmax_rows: bad argument");
  if (n_rows == 0) return AF_OK;
  argmax_rows_kernel<<<n_rows, 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(logits, vocab, tokens_out);
  return check_launch("argmax_rows_kernel");
}

extern "C" int af_embed_rows(const void* table, int32_t vocab, int32_t d_model, const int32_t* tokens, int32_t n_rows,
                             void* embeds_out, void* cuda_stream) {
  if (n_rows < 0 || vocab <= 0 || d_model <= 0 || (d_model % 8) || (n_rows > 0 && (!table || !tokens || !embeds_out)))
    return fail(AF_ERR_ARG, "af_embed_rows: bad argument (d_model must be a multiple of 8)");
  if ((reinterpret_cast<uintptr_t>(table) | reinterpret_cast<uintptr_t>(embeds_out)) & 15) return fail(AF_ERR_ARG, "af_embed_rows: pointers must be 16-byte aligned");
  if (n_rows == 0) return AF_OK;
  embed_rows_kernel<<<n_rows, 128, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(
      reinterpret_cast<const uint4*>(table), vocab, d_model / 8, tokens, reinterpret_cast<uint4*>(embeds_out));
  return check_launch("embed_rows_kernel");
}

extern "C" size_t af_gate_up_rows(int32_t ffn) { return ffn > 0 ? static_cast<size_t>((ffn + 63) / 64) * GEMM_BM : 0; }

extern "C" int af_prepare_gate_up(const void* gate, const void* up, void* dst, int32_t ffn, int32_t d_model, void* cuda_stream) {
  if (!gate || !up || !dst || ffn <= 0 || d_model <= 0 || (d_model % 8)) return fail(AF_ERR_ARG, "null pointer, or d_model not a multiple of 8");
  if ((reinterpret_cast<uintptr_t>(gate) | reinterpret_cast<uintptr_t>(up) | reinterpret_cast<uintptr_t>(dst)) & 15)
    return fail(AF_ERR_ARG, "pointers must be 16-byte aligned");
  const int vec_per_row = d_model / 8;
  const size_t n_vec = af_gate_up_rows(ffn) * vec_per_row;
  interleave_gate_up_kernel<<<static_cast<unsigned>((n_vec + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(
      reinterpret_cast<const uint4*>(gate), reinterpret_cast<const uint4*>(up), reinterpret_cast<uint4*>(dst), ffn, vec_per_row, n_vec);
  return check_launch("interleave_gate_up_kernel");
}

extern "C" int af_prepare_gate_up_fp8(const void* gate, const void* up, void* dst, int32_t ffn, int32_t d_model, void* cuda_stream) {
  if (!gate || !up || !dst || ffn <= 0 || d_model <= 0 || (d_model % 16)) return fail(AF_ERR_ARG, "null pointer, or d_model not a multiple of 16");
  if ((reinterpret_cast<uintptr_t>(gate) | reinterpret_cast<uintptr_t>(up) | reinterpret_cast<uintptr_t>(dst)) & 15)
    return fail(AF_ERR_ARG, "pointers must be 16-byte aligned");
  const int vec_per_row = d_model / 16;
  const size_t n_vec = af_gate_up_rows(ffn) * vec_per_row;
  interleave_gate_up_bytes_kernel<<<static_cast<unsigned>((n_vec + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(
      reinterpret_cast<const uint4*>(gate), reinterpret_cast<const uint4*>(up), reinterpret_cast<uint4*>(dst), ffn, vec_per_row, n_vec);
  return check_launch("interleave_gate_up_bytes_kernel");
}

extern "C" int af_debug_gemm_schedule(int32_t split_k, int32_t n_tile_pairs, int32_t n_kblocks, int32_t max_clusters,
                                      int32_t splits, int32_t* pieces, int32_t max_clusters_out) {
  if (!pieces) return fail(AF_ERR_ARG, "null output");
  std::vector<GemmPiece> flat;
  int n_cl = 0;
  const int rc = make_schedule(split_k == 3 ? SPLIT_K_SKEW : split_k == 2 ? SPLIT_SLABS : (split_k ? SPLIT_K : SPLIT_STREAMK), n_tile_pairs, n_kblocks, max_clusters, splits, &flat, &n_cl);
  if (rc) return rc;
  if (n_cl > max_clusters_out) return fail(AF_ERR_ARG, "%d clusters do not fit the output (%d)", n_cl, max_clusters_out);
  memcpy(pieces, flat.data(), flat.size() * sizeof(GemmPiece));
  return n_cl;
}

extern "C" int64_t af_debug_launch_count(void) { return g_launches.load(); }
extern "C" const char* af_last_error(void) { return g_err.c_str(); }

// ------------------------------------------------------------------------------------------------ the packed step
static int check_weights(const af_weights* w, bool need_lm) {
  if (!w || !w->layers) return fail(AF_ERR_ARG, "null weights");
  int rc = check_cfg(&w->cfg);
  if (rc) return rc;
  for (int l = 0; l < w->cfg.n_layers; ++l) {
    const af_layer_weights& L = w->layers[l];
    if (!L.wq || !L.wk || !L.wv || !L.wo || !L.w_gate || !L.w_up || !L.w_down || !L.g_attn || !L.g_mlp)
      return fail(AF_ERR_ARG, "null weight pointer in layer %d", l);
  }
  if (need_lm && (!w->g_final || !w->w_lm)) return fail(AF_ERR_ARG, "null g_final / w_lm");
  if (w->weight_format != AF_WEIGHTS_BF16 && w->weight_format != AF_WEIGHTS_FP16 && w->weight_format != AF_WEIGHTS_FP16_GU &&
      w->weight_format != AF_WEIGHTS_FP8)
    return fail(AF_ERR_ARG, "weight_format %d is not AF_WEIGHTS_BF16, AF_WEIGHTS_FP16, AF_WEIGHTS_FP16_GU or AF_WEIGHTS_FP8", w->weight_format);
  if (w->weight_format == AF_WEIGHTS_FP8) {
    if (!w->scales) return fail(AF_ERR_ARG, "AF_WEIGHTS_FP8 needs af_weights.scales");
    for (int l = 0; l < w->cfg.n_layers; ++l) {
      const af_layer_scales& S = w->scales[l];
      if (!S.sq || !S.sk || !S.sv || !S.so || !S.s_gate || !S.s_up || !S.s_down) return fail(AF_ERR_ARG, "null scale pointer in layer %d", l);
    }
  }
  return AF_OK;
}

// sta_dev != nullptr: the kernels ingest the segment table from that device struct (written by loop_advance_kernel, f1)
// instead of the by-value copy of `segs`; `segs` still drives validation, the host mirror and the launch geometry.
static int packed_forward_impl(const af_weights* w, const void* packed_embeds, const af_segment* segs, int32_t n_segs,
                               af_ring* g, float* hidden_out, void* workspace, size_t ws_bytes, void* cuda_stream,
                               const SegTableArg* sta_dev) {
  if (!g) return fail(AF_ERR_ARG, "null ring");
  if (n_segs < 0) return fail(AF_ERR_ARG, "n_segs < 0");
  if (n_segs == 0) { g->last_T = 0; return AF_OK; }  // legal no-op
  if (!segs) return fail(AF_ERR_ARG, "null segment table");
  if (n_segs > AF_MAX_SEGS) return fail(AF_ERR_SEGMENT, "%d segments > AF_MAX_SEGS", n_segs);
  int rc = check_weights(w, false);
  if (rc) return rc;
  const af_model_cfg& c = w->cfg;
  if (memcmp(&c, &g->cfg, sizeof c) != 0) return fail(AF_ERR_ARG, "weights cfg differs from the ring's cfg");
  const int R = g->rc.n_regions, C = g->rc.capacity;
  // ---- a0 validation on the host mirror, before any launch; same order of checks as the index model ----
  std::vector<char> seen(R, 0);
  long long T64 = 0;
  for (int s = 0; s < n_segs; ++s) {
    const af_segment& sg = segs[s];
    if (sg.req_id < 0 || sg.req_id >= R) return fail(AF_ERR_SEGMENT, "segment %d: req_id %d outside [0,%d)", s, sg.req_id, R);
    if (seen[sg.req_id]) return fail(AF_ERR_SEGMENT, "segment %d: req_id %d appears twice in one step", s, sg.req_id);
    seen[sg.req_id] = 1;
    if (sg.len < 1) return fail(AF_ERR_SEGMENT, "segment %d: len %d < 1", s, sg.len);
    if (sg.phase != AF_PHASE_PREFILL && sg.phase != AF_PHASE_DECODE) return fail(AF_ERR_SEGMENT, "segment %d: phase %d", s, sg.phase);
    if (sg.phase == AF_PHASE_DECODE && sg.len != 1) return fail(AF_ERR_SEGMENT, "segment %d: decode with len %d", s, sg.len);
    T64 += sg.len;
  }
  for (int s = 0; s < n_segs; ++s)
    if (segs[s].start_pos != g->len[segs[s].req_id])
      return fail(AF_ERR_POSITION, "segment %d: start_pos %d != current length %d of request %d", s, segs[s].start_pos,
                  g->len[segs[s].req_id], segs[s].req_id);
  for (int s = 0; s < n_segs; ++s) {
    const long long end = static_cast<long long>(segs[s].start_pos) + segs[s].len;
    if (g->window <= 0) {
      if (end > C) return fail(AF_ERR_CAPACITY, "segment %d: start_pos %d + len %d > capacity %d", s, segs[s].start_pos, segs[s].len, C);
    } else if (end > g->max_pos || (end > C && segs[s].len > C - g->window + 1)) {
      // f3: every row is appended before any row attends, so a wrapping segment's first row must keep its whole window
      return fail(AF_ERR_CAPACITY, "segment %d: start_pos %d + len %d exceeds max_pos %d, or wraps with len > capacity %d - window %d + 1",
                  s, segs[s].start_pos, segs[s].len, g->max_pos, C, g->window);
    }
  }
  if (T64 > g->max_rows) return fail(AF_ERR_CAPACITY, "%lld packed rows > ring rows %d", T64, g->max_rows);
  const int T = static_cast<int>(T64);
  if (!packed_embeds || !hidden_out) return fail(AF_ERR_ARG, "null embeds / hidden_out");
  if ((reinterpret_cast<uintptr_t>(packed_embeds) & 15) || (reinterpret_cast<uintptr_t>(hidden_out) & 15))
    return fail(AF_ERR_ARG, "embeds / hidden_out must be 16-byte aligned");
  Workspace ws;
  rc = carve(&c, workspace, ws_bytes, T, &ws);
  if (rc) return rc;

  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int D = c.d_model, F = c.ffn, H = c.n_heads, hd = c.head_dim;
  DevCtx* ctx = nullptr;
  if ((rc = get_ctx(&ctx))) return rc;
  if ((rc = serialise_on(ctx, st))) return rc;
  SegTableArg sta{};
  sta.n_segs = n_segs; sta.R = R; sta.C = C;
  int n_items = 0;
  for (int s = 0; s < n_segs; ++s) {
    sta.req[s] = segs[s].req_id; sta.start[s] = segs[s].start_pos; sta.len[s] = segs[s].len;
    sta.base[s] = g->base[segs[s].req_id];
    n_items += (segs[s].len + ATT_BQ - 1) / ATT_BQ;
  }
  cudaError_t le;
#define AF_LAUNCH(cat, name, ...)                                                                              \
  do {                                                                                                         \
    { ProfScope ps_(cat, st); le = launch_k1(__VA_ARGS__); }                                                   \
    if (le != cudaSuccess) return fail(AF_ERR_CUDA, "launch of %s failed: %s", name, cudaGetErrorString(le)); \
    if ((rc = check_launch(name))) return rc;                                                                  \
  } while (0)
  { ProfScope ps_(PC_OTHER, st);
  if (sta_dev) rowmap_dev_kernel<<<1, 256, 0, st>>>(sta_dev, g->tb, g->n_items_dev);
  else rowmap_kernel<<<1, 256, 0, st>>>(sta, g->tb, g->n_items_dev);
  }
  if ((rc = check_launch("rowmap_kernel"))) return rc;
  const float scale_log2 = 1.4426950408889634f / sqrtf(static_cast<float>(hd));
  const size_t layer_elems = static_cast<size_t>(2) * R * H * C * hd;
  // a4 on tcgen05 (attention_umma.cuh) when every segment's context fits one unit; attention_kernel otherwise
  bool att_umma = g_att_mode != 1 && hd == AU_HD && g->window == 0;
  int au_items = 0, au_rows = 0;
  for (int s = 0; s < n_segs; ++s) {
    if (segs[s].start_pos + segs[s].len > AU_KV_MAX) att_umma = false;
    if (segs[s].len == 1) ++au_rows;
    else au_items += (segs[s].len + AU_BQ - 1) / AU_BQ;
  }
  if (au_items > AU_MAX_ITEMS) att_umma = false;
  // default (mode 0): the units take the steps made of one-row segments only (decode-only steps: 2-4 % faster per step,
  // DESIGN.md 6.2b); a step with a multi-row segment is 1.5 % faster with attention_kernel as a kernel of its own
  if (g_att_mode == 0 && au_items > 0) att_umma = false;
  const int au_units = (au_items + au_rows) * H;
  auto attn_args = [&](int l) {
    AuArgs aa{};
    aa.q = ws.q_rot; aa.kv = g->kv + layer_elems * l; aa.out = ws.attn; aa.tb = g->tb; aa.n_segs = n_segs; aa.H = H; aa.R = R; aa.C = C;
    aa.scale_log2 = scale_log2; aa.sched = g->att_sched;
    if (g_trace && g_trace_att) {   // af_debug_trace(2): the attention units' stamps instead of the chain's
      aa.trace = g_trace + static_cast<size_t>(g_trace_n % TRACE_LAUNCHES) * GEMM_MAX_GRID * CH_TRACE_SLOTS;
      g_trace_meta[g_trace_n % TRACE_LAUNCHES] = {0, ctx->num_sms};
      ++g_trace_n;
    }
    return aa;
  };
  auto launch_attention = [&](int l) -> int {   // a4: segment-masked causal attention over the ring
    act_t* kvl = g->kv + layer_elems * l;
    if (att_umma) {
      const AuArgs aa = attn_args(l);
      AF_LAUNCH(PC_ATTENTION, "attention_umma_kernel", attention_umma_kernel, dim3(au_units < ctx->num_sms ? au_units : ctx->num_sms),
                dim3(AU_THREADS), static_cast<size_t>(AU_SMEM_BYTES), st, aa);
      return AF_OK;
    }
    auto att = hd == 128 ? (g->window > 0 ? attention_kernel<128, true> : attention_kernel<128, false>)
                         : (g->window > 0 ? attention_kernel<64, true> : attention_kernel<64, false>);
    AF_LAUNCH(PC_ATTENTION, "attention_kernel", att, dim3(H, n_items), dim3(ATT_THREADS), att_smem_bytes(hd), st,
              static_cast<const act_t*>(ws.q_rot), static_cast<const act_t*>(kvl), ws.attn, g->tb, H, R, C, scale_log2,
              g->window);
    return AF_OK;
  };
  // ---- the layer chain (chain.cuh): per layer ONE persistent launch for every projection and row stage + attention ----
  const bool fp8 = w->weight_format == AF_WEIGHTS_FP8;
  // every work list of the chain is built (and cached) BEFORE the first launch: a shape it cannot schedule falls back to the
  // per-stage path (FP8: AF_ERR_UNSUPPORTED) with nothing enqueued
  const int t_chunks = T > GEMM_MAX_TOK ? 2 : 1;
  auto chain_schedulable = [&]() {
    const int kd = (D + GEMM_BK - 1) / GEMM_BK, kf = (F + GEMM_BK - 1) / GEMM_BK;
    const int d_pairs = ((D + GEMM_BM - 1) / GEMM_BM + 1) / 2, gu_pairs = ((F + 63) / 64 + 1) / 2;
    const int o_splits = gemm_split_count(ctx, (D + GEMM_BM - 1) / GEMM_BM, D);
    Sched sc;
    return build_schedule(ctx, SPLIT_SLABS, (3 * ((D + GEMM_BM - 1) / GEMM_BM) + 1) / 2, kd, ctx->max_clusters, QKV_MAX_SLABS, &sc, t_chunks) == AF_OK &&
           build_schedule(ctx, (o_splits > 1 && kd >= 4 * o_splits) ? SPLIT_K_SKEW : SPLIT_K, d_pairs, kd, ctx->max_clusters, o_splits, &sc, t_chunks) == AF_OK &&
           build_schedule(ctx, SPLIT_K, d_pairs, kf, ctx->max_clusters, gemm_split_count(ctx, (D + GEMM_BM - 1) / GEMM_BM, F), &sc, t_chunks) == AF_OK &&
           build_schedule(ctx, SPLIT_STREAMK, gu_pairs, kd, ctx->max_clusters, 1, &sc, t_chunks) == AF_OK;
  };
  if (fp8 && (T > 2 * GEMM_MAX_TOK || D > 4096 || D % 256 != 0 || F < 128 || ctx->max_clusters < 2 || g_prof_stages))
    return fail(AF_ERR_UNSUPPORTED, "AF_WEIGHTS_FP8 runs on the layer chain only: T <= %d packed rows, d_model <= 4096 and a multiple of 256", 2 * GEMM_MAX_TOK);
  if (fp8 && !chain_schedulable()) return fail(AF_ERR_UNSUPPORTED, "AF_WEIGHTS_FP8: this shape has no layer-chain schedule on this device");
  const bool use_chain = (w->weight_format == AF_WEIGHTS_FP16_GU || fp8) && T <= 2 * GEMM_MAX_TOK && D <= 4096 && D % 256 == 0 && F >= 128 &&
                         ctx->max_clusters >= 2 && !g_prof_stages && chain_schedulable();
  if (use_chain) {
    StreamCtx sctx;
    if ((rc = get_stream_ctx(ctx, st, &sctx))) return rc;
    const long long split_stride = static_cast<long long>(ws.max_rows) * D;
    const long long qkv_stride = static_cast<long long>(ws.max_rows) * 3 * D;
    auto begin = [&](ChainBuilder& b) {
      b.ctx = ctx; b.max_rows = ws.max_rows; b.fp8 = fp8;
      int Tc = T;                                               // rows of one token chunk
      b.a.T0 = 0;
      if (T > GEMM_MAX_TOK) { Tc = ((T + 1) / 2 + 15) / 16 * 16; b.a.T0 = Tc; b.chunks = 2; }
      int n_pad = (Tc + 15) / 16 * 16;
      if (n_pad <= 256) { b.a.n1 = n_pad; b.a.n2 = 0; }
      else { b.a.n1 = ((Tc + 1) / 2 + 15) / 16 * 16; b.a.n2 = b.a.n1; }
      b.a.T = T; b.a.D = D; b.a.eps = c.rms_eps; b.a.x = hidden_out; b.a.bar = sctx.bar; b.a.flags = sctx.flags;
      b.a.partial = reinterpret_cast<uint8_t*>(ws.partial); b.a.tb = g->tb; b.a.rope_tab = g->rope_tab;
      b.a.H = H; b.a.hd = hd; b.a.R = R; b.a.C = C;
    };
    auto add_qkv_rope = [&](ChainBuilder& b, int l) -> int {
      const af_layer_weights& L = w->layers[l];
      const void* wqkv[3] = {L.wq, L.wk, L.wv};
      const float* sqkv[3] = {fp8 ? w->scales[l].sq : nullptr, fp8 ? w->scales[l].sk : nullptr, fp8 ? w->scales[l].sv : nullptr};
      const int* pair_slabs = nullptr;
      int r = chain_add_gemm(b, wqkv, sqkv, 3, D, 0, D, SPLIT_SLABS, QKV_MAX_SLABS, EPI_STORE, ws.xn, ws.qkv, 3LL * D, qkv_stride, D, &pair_slabs, nullptr);
      if (r) return r;
      return chain_add_rope(b, ws.qkv, qkv_stride, pair_slabs, ws.q_rot, g->kv + layer_elems * l);
    };
    {   // launch 0: x = embeds; xn = RMSNorm(x; g_attn[0]) | QKV of layer 0 | RoPE + ring append
      ChainBuilder b;
      begin(b);
      if ((rc = chain_add_rows(b, packed_embeds, 1, 0, 0, w->layers[0].g_attn, ws.xn))) return rc;
      if ((rc = add_qkv_rope(b, 0))) return rc;
      if (att_umma && (rc = chain_add_attn(b, attn_args(0)))) return rc;
      if ((rc = chain_launch(b, st, PC_CHAIN))) return rc;
    }
    for (int l = 0; l < c.n_layers; ++l) {
      if (!att_umma && (rc = launch_attention(l))) return rc;   // (else: the last phase of the previous launch)
      const af_layer_weights& L = w->layers[l];
      ChainBuilder b;
      begin(b);
      int n_slabs = 0;
      const void* wo[3] = {L.wo, nullptr, nullptr};
      const float* so[3] = {fp8 ? w->scales[l].so : nullptr, nullptr, nullptr};
      const float* sgu[3] = {fp8 ? w->scales[l].s_gate : nullptr, fp8 ? w->scales[l].s_up : nullptr, nullptr};
      const float* sd[3] = {fp8 ? w->scales[l].s_down : nullptr, nullptr, nullptr};
      if ((rc = chain_add_gemm(b, wo, so, 1, D, 0, D, SPLIT_K, GEMM_MAX_SPLITS, EPI_STORE, ws.attn, reinterpret_cast<act_t*>(ws.split), D, split_stride, D, nullptr, &n_slabs))) return rc;
      if ((rc = chain_add_rows(b, ws.split, 0, n_slabs, split_stride, L.g_mlp, ws.xn))) return rc;
      const void* wgu[3] = {L.w_gate, nullptr, nullptr};
      if ((rc = chain_add_gemm(b, wgu, sgu, 2, F, 2, D, SPLIT_STREAMK, 1, EPI_SWIGLU, ws.xn, ws.h, F, 0, F, nullptr, nullptr))) return rc;
      const void* wd[3] = {L.w_down, nullptr, nullptr};
      if ((rc = chain_add_gemm(b, wd, sd, 1, D, 0, F, SPLIT_K, GEMM_MAX_SPLITS, EPI_STORE, ws.h, reinterpret_cast<act_t*>(ws.split), D, split_stride, D, nullptr, &n_slabs))) return rc;
      if (l + 1 < c.n_layers) {
        if ((rc = chain_add_rows(b, ws.split, 0, n_slabs, split_stride, w->layers[l + 1].g_attn, ws.xn))) return rc;
        if ((rc = add_qkv_rope(b, l + 1))) return rc;
        if (att_umma && (rc = chain_add_attn(b, attn_args(l + 1)))) return rc;
      } else {
        if ((rc = chain_add_rows(b, ws.split, 0, n_slabs, split_stride, nullptr, nullptr))) return rc;   // hidden_out: no final norm
      }
      if ((rc = chain_launch(b, st, PC_CHAIN))) return rc;
    }
    for (int s = 0; s < n_segs; ++s) g->len[segs[s].req_id] = segs[s].start_pos + segs[s].len;   // a9 ring commit
    g->last_T = T;
    return serialise_done(ctx, st);
  }
  // ---- the per-stage path (bf16 / unpacked weights, T > 512, or per-stage profiling): one kernel per stage ----
  {
    const size_t n = static_cast<size_t>(T) * D;
    AF_LAUNCH(PC_OTHER, "embed_to_residual_kernel", embed_to_residual_kernel,
              dim3(static_cast<unsigned>((n / 4 + 255) / 256)), dim3(256), 0, st,
              reinterpret_cast<const __nv_bfloat16*>(packed_embeds), hidden_out, n);
  }
  const int row_threads = row_threads_for(D);
  const int wfmt = w->weight_format == AF_WEIGHTS_FP16 || w->weight_format == AF_WEIGHTS_FP16_GU;
  const bool gu_packed = w->weight_format == AF_WEIGHTS_FP16_GU;
  const long long split_stride = static_cast<long long>(ws.max_rows) * D;
  int prev_splits = 0;   // split-K slabs of the previous projection still to be added to the residual stream
  auto split_count = [&](int n_tiles, int K) { return gemm_split_count(ctx, n_tiles, K); };
  const int d_tiles = (D + GEMM_BM - 1) / GEMM_BM;
  for (int l = 0; l < c.n_layers; ++l) {
    const af_layer_weights& L = w->layers[l];
    act_t* kvl = g->kv + layer_elems * l;
    // a8(prev) + a1: x += down partials; xn = RMSNorm(x; g_attn)
    AF_LAUNCH(PC_RMSNORM, "residual_norm_kernel", residual_norm_kernel, dim3(T), dim3(row_threads), 0, st, hidden_out,
              reinterpret_cast<const act_t*>(ws.split), prev_splits, split_stride,
              reinterpret_cast<const __nv_bfloat16*>(L.g_attn), ws.xn, D, c.rms_eps);
    // a2: QKV projection (stream-K with fix-up, fp16 q|k|v rows)
    {
      GemmParams gp{};
      gp.part_f16 = 1; gp.w_fp16 = wfmt; gp.n_parts = 3; gp.part_rows = D; gp.a_pair = 0; gp.K = D; gp.split = SPLIT_STREAMK; gp.epi = EPI_STORE;
      gp.partial = ws.partial;
      const OutView ov{ws.qkv, -2, D, 3, T, D, 3LL * D, 32};
      const void* wqkv[3] = {L.wq, L.wk, L.wv};
      if ((rc = launch_gemm(PC_GEMM_QKV, st, gp, ov, ws.xn, ws.max_rows, wqkv, T))) return rc;
    }
    // a3: FusedRoPEAndWriteKV (Alg. 2 l.3): rotate q, k at the row's position; k, v go straight to the ring slot
    AF_LAUNCH(PC_ROPE_APPEND, "rope_append_kernel", rope_append_kernel, dim3(T), dim3(row_threads), 0, st,
              static_cast<const act_t*>(ws.qkv), ws.q_rot, kvl, static_cast<const float2*>(g->rope_tab), g->tb,
              H, hd, R, C);
    if ((rc = launch_attention(l))) return rc;
    // a5: O projection, split-K slabs (added to the residual by the next kernel)
    {
      GemmParams gp{};
      gp.w_fp16 = wfmt; gp.n_parts = 1; gp.part_rows = D; gp.K = D; gp.split = SPLIT_K; gp.epi = EPI_STORE; gp.partial = ws.partial;
      const OutView ov{ws.split, -2, D, GEMM_MAX_SPLITS, T, split_stride, D, 32};
      const void* wo[3] = {L.wo, nullptr, nullptr};
      if ((rc = launch_gemm(PC_GEMM_O, st, gp, ov, ws.attn, ws.max_rows, wo, T))) return rc;
      prev_splits = split_count(d_tiles, D);
    }
    // a5 residual + a6: x += O partials; xn = RMSNorm(x; g_mlp)
    AF_LAUNCH(PC_RMSNORM, "residual_norm_kernel", residual_norm_kernel, dim3(T), dim3(row_threads), 0, st, hidden_out,
              reinterpret_cast<const act_t*>(ws.split), prev_splits, split_stride,
              reinterpret_cast<const __nv_bfloat16*>(L.g_mlp), ws.xn, D, c.rms_eps);
    // a7: gate/up projection with the fused SiLU*mul epilogue
    {
      GemmParams gp{};
      gp.part_f16 = 1; gp.w_fp16 = wfmt; gp.n_parts = 2; gp.part_rows = F; gp.a_pair = gu_packed ? 2 : 1; gp.K = D; gp.split = SPLIT_STREAMK; gp.epi = EPI_SWIGLU;
      gp.partial = ws.partial;
      const OutView ov{ws.h, -2, F, 1, T, F, F, 16};
      const void* wgu[3] = {L.w_gate, gu_packed ? L.w_gate : L.w_up, nullptr};
      if ((rc = launch_gemm(PC_GEMM_GATEUP, st, gp, ov, ws.xn, ws.max_rows, wgu, T))) return rc;
    }
    // a8: down projection, split-K slabs
    {
      GemmParams gp{};
      gp.w_fp16 = wfmt; gp.n_parts = 1; gp.part_rows = D; gp.K = F; gp.split = SPLIT_K; gp.epi = EPI_STORE; gp.partial = ws.partial;
      const OutView ov{ws.split, -2, D, GEMM_MAX_SPLITS, T, split_stride, D, 32};
      const void* wd[3] = {L.w_down, nullptr, nullptr};
      if ((rc = launch_gemm(PC_GEMM_DOWN, st, gp, ov, ws.h, ws.max_rows, wd, T))) return rc;
      prev_splits = split_count(d_tiles, F);
    }
  }
  // a8 of the last layer: x += down partials (no norm: hidden_out is the pre-final-norm residual stream)
  AF_LAUNCH(PC_RMSNORM, "residual_norm_kernel", residual_norm_kernel, dim3(T), dim3(row_threads), 0, st, hidden_out,
            reinterpret_cast<const act_t*>(ws.split), prev_splits, split_stride, static_cast<const __nv_bfloat16*>(nullptr),
            static_cast<act_t*>(nullptr), D, c.rms_eps);
#undef AF_LAUNCH
  // ---- a9 ring commit: a relabelling, zero bytes moved (replaces InPlaceShiftKV) ----
  for (int s = 0; s < n_segs; ++s) g->len[segs[s].req_id] = segs[s].start_pos + segs[s].len;
  g->last_T = T;
  return serialise_done(ctx, st);
}

extern "C" int af_packed_forward(const af_weights* w, const void* packed_embeds, const af_segment* segs, int32_t n_segs,
                                 af_ring* g, float* hidden_out, void* workspace, size_t ws_bytes, void* cuda_stream) {
  return packed_forward_impl(w, packed_embeds, segs, n_segs, g, hidden_out, workspace, ws_bytes, cuda_stream, nullptr);
}

extern "C" int af_logits_rows(const af_weights* w, const float* hidden, const int32_t* rows, int32_t n_rows,
                              float* logits_out, void* workspace, size_t ws_bytes, void* cuda_stream) {
  int rc = check_weights(w, true);
  if (rc) return rc;
  if (n_rows == 0) return AF_OK;
  if (!hidden || !rows || !logits_out || n_rows < 0) return fail(AF_ERR_ARG, "null/negative argument");
  if (n_rows > 256) return fail(AF_ERR_UNSUPPORTED, "n_rows %d > 256", n_rows);
  for (int i = 0; i < n_rows; ++i)
    if (rows[i] < 0) return fail(AF_ERR_ARG, "rows[%d] = %d < 0", i, rows[i]);
  const af_model_cfg& c = w->cfg;
  Workspace ws;
  rc = carve(&c, workspace, ws_bytes, n_rows, &ws);
  if (rc) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  RowListArg rl{};
  for (int i = 0; i < n_rows; ++i) rl.rows[i] = rows[i];
  {
    ProfScope ps_(PC_RMSNORM, st);
    cudaError_t le = launch_k1(gather_norm_kernel, dim3(n_rows), dim3(row_threads_for(c.d_model)), 0, st, rl, hidden,
                              reinterpret_cast<const __nv_bfloat16*>(w->g_final), ws.xn, c.d_model, c.rms_eps);
    if (le != cudaSuccess) return fail(AF_ERR_CUDA, "launch of gather_norm_kernel failed: %s", cudaGetErrorString(le));
  }
  if ((rc = check_launch("gather_norm_kernel"))) return rc;
  GemmParams gp{};
  gp.w_fp16 = w->weight_format != AF_WEIGHTS_BF16;   // (AF_WEIGHTS_FP8: the LM head stays a prepared fp16 matrix)
  gp.n_parts = 1; gp.part_rows = c.vocab; gp.K = c.d_model; gp.split = SPLIT_STREAMK; gp.epi = EPI_STORE;
  gp.partial = ws.partial;
  if (c.vocab % 4) return fail(AF_ERR_UNSUPPORTED, "vocab must be a multiple of 4 (16-byte logits rows)");
  const OutView ov{logits_out, 4, c.vocab, 1, n_rows, c.vocab, c.vocab, 32};
  const void* wl[3] = {w->w_lm, nullptr, nullptr};
  return launch_gemm(PC_GEMM_LM, st, gp, ov, ws.xn, ws.max_rows, wl, n_rows);
}

extern "C" int af_debug_gemm(const void* a, const void* wmat, float* out, int32_t n_tok, int32_t n_out, int32_t k,
                             void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (!a || !wmat || !out || !workspace) return fail(AF_ERR_ARG, "null argument");
  if (n_tok <= 0 || n_out <= 0 || k <= 0 || (k % 8)) return fail(AF_ERR_ARG, "bad GEMM shape");
  if (ws_bytes < gemm_partial_bytes()) return fail(AF_ERR_WORKSPACE, "workspace < %zu bytes", gemm_partial_bytes());
  GemmParams gp{};
  gp.n_parts = 1; gp.part_rows = n_out; gp.K = k; gp.split = SPLIT_STREAMK; gp.epi = EPI_STORE;
  gp.partial = workspace;
  if (n_out % 4) return fail(AF_ERR_ARG, "n_out must be a multiple of 4");
  const OutView ov{out, 4, n_out, 1, n_tok, n_out, n_out, 32};
  const void* wl[3] = {wmat, nullptr, nullptr};
  return launch_gemm(PC_OTHER, reinterpret_cast<cudaStream_t>(cuda_stream), gp, ov, a, n_tok, wl, n_tok);
}

// ------------------------------------------------------------------------------------------------ f1: Alg. 1 on the device
// The pipeline loop of Algorithm 1 with its state on the device: segment table and ring bookkeeping
// advanced by loop_advance_kernel, ArgMax -> Embed feedback through af_argmax_rows / af_embed_rows' kernels,
// A_sequences kept by loop_commit_kernel.  The host only mirrors the integer schedule (validation, launch geometry)
// and, once the pipeline is full, replays ONE captured CUDA graph per step: no host synchronisation anywhere.
struct af_loop {
  af_weights w;
  af_ring* g;
  const void* table;
  int L_P, K, t;
  void* ws; size_t ws_bytes;
  uint8_t* mem;
  LoopState* ls; SegTableArg* sta;
  __nv_bfloat16* packed; float* hidden; float* logits; int* tok;
  int steady_direct;            // steady-shape steps issued as plain launches (the first one warms every host cache)
  cudaGraphExec_t graph; int64_t graph_nodes;
};

extern "C" int af_loop_create(const af_weights* w, af_ring* g, const void* embed_table, int32_t prefill_len, int32_t chunk_k,
                              void* workspace, size_t ws_bytes, af_loop** out) {
  if (!g || !out || !embed_table) return fail(AF_ERR_ARG, "null argument");
  int rc = check_weights(w, true);
  if (rc) return rc;
  if (memcmp(&w->cfg, &g->cfg, sizeof w->cfg) != 0) return fail(AF_ERR_ARG, "weights cfg differs from the ring's cfg");
  if (reinterpret_cast<uintptr_t>(embed_table) & 15) return fail(AF_ERR_ARG, "embed_table must be 16-byte aligned");
  const int R = g->rc.n_regions, C = g->rc.capacity, K = chunk_k, L_P = prefill_len;
  if (K < 1 || K > AF_MAX_SEGS || L_P < 1) return fail(AF_ERR_ARG, "need 1 <= chunk_k <= %d and prefill_len >= 1", AF_MAX_SEGS);
  if (R < K || R > AF_MAX_SEGS) return fail(AF_ERR_SEGMENT, "the pipeline needs chunk_k <= n_regions <= %d (K = %d, R = %d)", AF_MAX_SEGS, K, R);
  if (L_P + K - 1 > C) return fail(AF_ERR_CAPACITY, "prefill_len %d + chunk_k %d - 1 > capacity %d", L_P, K, C);
  const int T = L_P + K - 1;
  if (T > g->max_rows) return fail(AF_ERR_CAPACITY, "%d packed rows > ring rows %d", T, g->max_rows);
  Workspace wsp;
  if ((rc = carve(&w->cfg, workspace, ws_bytes, T, &wsp))) return rc;
  const size_t D = w->cfg.d_model, V = w->cfg.vocab;
  size_t off = 0;
  auto take = [&](size_t n) { const size_t o = off; off += align_up(n, 256); return o; };
  const size_t o_ls = take(sizeof(LoopState)), o_sta = take(sizeof(SegTableArg)), o_pk = take(T * D * 2),
               o_hid = take(T * D * 4), o_lg = take(K * V * 4), o_tok = take(AF_MAX_SEGS * sizeof(int));
  af_loop* lp = new af_loop();
  cudaError_t e = cudaMalloc(&lp->mem, off);
  if (e != cudaSuccess) { delete lp; return fail(AF_ERR_CUDA, "cudaMalloc: %s", cudaGetErrorString(e)); }
  lp->w = *w; lp->g = g; lp->table = embed_table; lp->L_P = L_P; lp->K = K; lp->t = 0;
  lp->ws = workspace; lp->ws_bytes = ws_bytes;
  lp->ls = reinterpret_cast<LoopState*>(lp->mem + o_ls); lp->sta = reinterpret_cast<SegTableArg*>(lp->mem + o_sta);
  lp->packed = reinterpret_cast<__nv_bfloat16*>(lp->mem + o_pk); lp->hidden = reinterpret_cast<float*>(lp->mem + o_hid);
  lp->logits = reinterpret_cast<float*>(lp->mem + o_lg); lp->tok = reinterpret_cast<int*>(lp->mem + o_tok);
  lp->steady_direct = 0; lp->graph = nullptr; lp->graph_nodes = 0;
  // every region starts empty at its current rotation; the device state starts as a copy of the host mirror
  LoopState* h = new LoopState();
  memset(h, 0, sizeof *h);
  h->L_P = L_P; h->K = K; h->R = R; h->C = C; h->frame_id = -1;
  for (int r = 0; r < R; ++r) { g->len[r] = 0; h->base[r] = g->base[r]; }
  for (int s = 0; s < AF_MAX_SEGS; ++s) h->frame_tok[s] = -1;
  e = cudaMemset(lp->mem, 0, off);
  if (e == cudaSuccess) e = cudaMemcpy(lp->ls, h, sizeof *h, cudaMemcpyHostToDevice);
  delete h;
  if (e != cudaSuccess) { cudaFree(lp->mem); delete lp; return fail(AF_ERR_CUDA, "loop state upload: %s", cudaGetErrorString(e)); }
  *out = lp;
  return AF_OK;
}

extern "C" int af_loop_destroy(af_loop* lp) {
  if (!lp) return AF_OK;
  if (lp->graph) cudaGraphExecDestroy(lp->graph);
  cudaFree(lp->mem);
  delete lp;
  return AF_OK;
}

extern "C" int af_loop_buffers(af_loop* lp, void** prefill_embeds, float** hidden, float** logits, int32_t** tokens,
                               int32_t** frame) {
  if (!lp) return fail(AF_ERR_ARG, "null loop");
  if (prefill_embeds) *prefill_embeds = lp->packed;
  if (hidden) *hidden = lp->hidden;
  if (logits) *logits = lp->logits;
  if (tokens) *tokens = lp->tok;
  if (frame) *frame = &lp->ls->frame_id;
  return AF_OK;
}

// the launches of one pipeline step, in stream order (also what the graph captures)
static int loop_enqueue(af_loop* lp, const af_segment* segs, int n_dec, cudaStream_t st) {
  const af_model_cfg& c = lp->w.cfg;
  int rc;
  loop_advance_kernel<<<1, 32, 0, st>>>(lp->ls, lp->sta);
  if ((rc = check_launch("loop_advance_kernel"))) return rc;
  if (n_dec > 0) {   // Alg. 1 l.2: decode row of stage s = Embed(token stage s-1 produced in the previous step)
    embed_rows_kernel<<<n_dec, 128, 0, st>>>(reinterpret_cast<const uint4*>(lp->table), c.vocab, c.d_model / 8, lp->tok,
                                             reinterpret_cast<uint4*>(lp->packed + static_cast<size_t>(lp->L_P) * c.d_model));
    if ((rc = check_launch("embed_rows_kernel"))) return rc;
  }
  if ((rc = packed_forward_impl(&lp->w, lp->packed, segs, 1 + n_dec, lp->g, lp->hidden, lp->ws, lp->ws_bytes, st, lp->sta))) return rc;
  int32_t rows[AF_MAX_SEGS];
  for (int s = 0; s <= n_dec; ++s) rows[s] = lp->L_P - 1 + s;   // prediction rows: last prefill row, then the decode rows
  if ((rc = af_logits_rows(&lp->w, lp->hidden, rows, 1 + n_dec, lp->logits, lp->ws, lp->ws_bytes, st))) return rc;
  argmax_rows_kernel<<<1 + n_dec, 256, 0, st>>>(lp->logits, c.vocab, lp->tok);
  if ((rc = check_launch("argmax_rows_kernel"))) return rc;
  loop_commit_kernel<<<1, 32, 0, st>>>(lp->ls, lp->tok);
  return check_launch("loop_commit_kernel");
}

extern "C" int af_loop_step(af_loop* lp, int32_t use_graph, void* cuda_stream) {
  if (!lp) return fail(AF_ERR_ARG, "null loop");
  af_ring* g = lp->g;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int R = g->rc.n_regions, K = lp->K, L_P = lp->L_P, t = lp->t;
  const int n_dec = t < K - 1 ? t : K - 1;
  // host mirror of loop_advance_kernel (same integer rules; the device computes its own copy)
  int rc = af_ring_reset_slot(g, t % R, -1);
  if (rc) return rc;
  af_segment segs[AF_MAX_SEGS];
  segs[0] = af_segment{t % R, AF_PHASE_PREFILL, 0, L_P};
  for (int s = 1; s <= n_dec; ++s) segs[s] = af_segment{(t - s) % R, AF_PHASE_DECODE, g->len[(t - s) % R], 1};
  const bool steady = n_dec == K - 1;
  const bool graph_ok = steady && use_graph && st != nullptr && !g_prof_on && !g_trace;
  if (graph_ok && lp->graph) {
    cudaError_t e = cudaGraphLaunch(lp->graph, st);
    if (e != cudaSuccess) return fail(AF_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(e));
    g_launches.fetch_add(lp->graph_nodes, std::memory_order_relaxed);
    for (int s = 0; s <= n_dec; ++s) g->len[segs[s].req_id] = segs[s].start_pos + segs[s].len;   // a9 on the mirror
    g->last_T = L_P + n_dec;
    lp->t = t + 1;
    return AF_OK;
  }
  // the first steady step runs as plain launches (it fills the schedule / tensor-map caches, which allocate); the
  // second is captured, instantiated and launched; every later one is a replay
  const bool capture = graph_ok && lp->steady_direct >= 1;
  if (capture) {
    cudaError_t e = cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) return fail(AF_ERR_CUDA, "cudaStreamBeginCapture: %s", cudaGetErrorString(e));
  }
  rc = loop_enqueue(lp, segs, n_dec, st);
  if (capture) {
    cudaGraph_t gr = nullptr;
    cudaError_t e = cudaStreamEndCapture(st, &gr);
    if (rc) { if (gr) cudaGraphDestroy(gr); return rc; }
    if (e != cudaSuccess) return fail(AF_ERR_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    size_t n_nodes = 0;
    cudaGraphGetNodes(gr, nullptr, &n_nodes);
    e = cudaGraphInstantiate(&lp->graph, gr, 0);
    cudaGraphDestroy(gr);
    if (e != cudaSuccess) { lp->graph = nullptr; return fail(AF_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e)); }
    lp->graph_nodes = static_cast<int64_t>(n_nodes);
    e = cudaGraphLaunch(lp->graph, st);
    if (e != cudaSuccess) return fail(AF_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(e));
  }
  if (rc) return rc;
  if (steady) ++lp->steady_direct;
  lp->t = t + 1;
  return AF_OK;
}

extern "C" int32_t af_loop_steps_done(const af_loop* lp) { return lp ? lp->t : -1; }

// ------------------------------------------------------------------------------------------------ f1 without allocation
// af_argmax_rows_static: the ArgMax of Alg. 1 l.5/l.8 for callers that cannot allocate (code under stream capture, tight
// serving loops).  A variant of argmax_rows_kernel that splits every row's vocabulary over several CTAs (a decode step
// has 1 + n_dec rows: one CTA per row leaves most of the 148 SMs idle) and therefore needs scratch: the per-chunk
// (value, index) candidates and one arrival ticket per row.  That scratch is the file-scope array below - 131 KB that
// every GPU which loads the library holds until exit - instead of caller or cudaMalloc memory.  In HOST code the array's
// name is a host-side stand-in, not a device address: the launch takes the pointer cudaGetSymbolAddress returns, looked
// up once per device with that device current.
constexpr int ARGMAX_STATIC_MAX_ROWS = AF_ARGMAX_STATIC_MAX_ROWS;
constexpr int ARGMAX_STATIC_MAX_CHUNKS = 64;       // CTAs per row at most
constexpr int ARGMAX_STATIC_MIN_CHUNK = 2048;      // logits per CTA at least (8 per thread)
constexpr int ARGMAX_STATIC_MAX_DEVICES = 64;
struct ArgmaxScratch {
  float v[ARGMAX_STATIC_MAX_ROWS][ARGMAX_STATIC_MAX_CHUNKS];
  int i[ARGMAX_STATIC_MAX_ROWS][ARGMAX_STATIC_MAX_CHUNKS];
  unsigned ticket[ARGMAX_STATIC_MAX_ROWS];         // chunks of the row that have published their candidate; 0 between calls
};
static __device__ __align__(256) unsigned char g_argmax_scratch[sizeof(ArgmaxScratch)];

// grid (n_chunks, n_rows).  CTA (c, r) reduces logits[r, c*chunk .. (c+1)*chunk) with argmax_rows_kernel's order-free
// rule ("greater value, or equal value and lower index, wins"; NaNs lose every comparison), publishes its candidate and
// takes a ticket; the CTA that takes the row's last ticket reduces the candidates, stores the token and puts the ticket
// back to 0.
__global__ void __launch_bounds__(256)
argmax_rows_split_kernel(const float* __restrict__ logits, int vocab, int chunk, int* __restrict__ tokens_out, ArgmaxScratch* sc) {
  __shared__ float s_v[8];
  __shared__ int s_i[8];
  __shared__ bool s_last;
  const int r = blockIdx.y, c = blockIdx.x, n_chunks = gridDim.x;
  const float* row = logits + static_cast<size_t>(r) * vocab;
  const int v0 = c * chunk, v1 = min(vocab, v0 + chunk);
  auto better = [](float a, int ai, float b, int bi) { return a > b || (a == b && ai < bi); };
  auto block_reduce = [&](float& best, int& best_i) {   // result in thread 0
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ov = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, best_i, o);
      if (better(ov, oi, best, best_i)) { best = ov; best_i = oi; }
    }
    if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = best; s_i[threadIdx.x >> 5] = best_i; }
    __syncthreads();
    if (threadIdx.x == 0)
      for (int w = 1; w < 8; ++w)
        if (better(s_v[w], s_i[w], best, best_i)) { best = s_v[w]; best_i = s_i[w]; }
  };
  float best = -INFINITY;
  int best_i = 0x7fffffff;
  for (int v = v0 + threadIdx.x; v < v1; v += 256) {
    const float x = row[v];
    if (better(x, v, best, best_i)) { best = x; best_i = v; }
  }
  block_reduce(best, best_i);
  if (threadIdx.x == 0) {
    sc->v[r][c] = best;
    sc->i[r][c] = best_i;
    __threadfence();                                     // the candidate is visible before the ticket is
    s_last = atomicAdd(&sc->ticket[r], 1u) == static_cast<unsigned>(n_chunks - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();                                       // the other chunks' candidates, published before their tickets
  best = -INFINITY;
  best_i = 0x7fffffff;
  if (threadIdx.x < n_chunks) {
    best = __ldcg(&sc->v[r][threadIdx.x]);
    best_i = __ldcg(&sc->i[r][threadIdx.x]);
  }
  __syncthreads();                                       // s_v / s_i are reused
  block_reduce(best, best_i);
  if (threadIdx.x == 0) {
    tokens_out[r] = best_i == 0x7fffffff ? 0 : best_i;
    sc->ticket[r] = 0u;
  }
}

static std::mutex g_argmax_static_mu;
static ArgmaxScratch* g_argmax_static_ptr[ARGMAX_STATIC_MAX_DEVICES] = {};

extern "C" int af_argmax_rows_static(const float* logits, int32_t n_rows, int32_t vocab, int32_t* tokens_out, void* cuda_stream) {
  if (n_rows < 0 || vocab <= 0 || (n_rows > 0 && (!logits || !tokens_out))) return fail(AF_ERR_ARG, "af_argmax_rows_static: bad argument");
  if (n_rows > ARGMAX_STATIC_MAX_ROWS)
    return fail(AF_ERR_UNSUPPORTED, "af_argmax_rows_static: n_rows %d > %d, the rows its static scratch holds (use af_argmax_rows)", n_rows, ARGMAX_STATIC_MAX_ROWS);
  if (n_rows == 0) return AF_OK;
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= ARGMAX_STATIC_MAX_DEVICES) return fail(AF_ERR_UNSUPPORTED, "af_argmax_rows_static: device %d outside [0,%d)", dev, ARGMAX_STATIC_MAX_DEVICES);
  ArgmaxScratch* sc = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_argmax_static_mu);
    if (!g_argmax_static_ptr[dev]) {                     // set-up, once per device, with that device current
      void* p = nullptr;
      CUDA_TRY(cudaGetSymbolAddress(&p, g_argmax_scratch));
      g_argmax_static_ptr[dev] = static_cast<ArgmaxScratch*>(p);
    }
    sc = g_argmax_static_ptr[dev];
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  int n_chunks = (vocab + ARGMAX_STATIC_MIN_CHUNK - 1) / ARGMAX_STATIC_MIN_CHUNK;
  if (n_chunks > ARGMAX_STATIC_MAX_CHUNKS) n_chunks = ARGMAX_STATIC_MAX_CHUNKS;
  const int chunk = (vocab + n_chunks - 1) / n_chunks;
  n_chunks = (vocab + chunk - 1) / chunk;                // no empty chunk
  // the array keeps the last call's contents: tickets must start at 0 (they do after a call that ran to its end; a call
  // that was aborted, or one that overlapped another, may have left some behind)
  CUDA_TRY(cudaMemsetAsync(sc->ticket, 0, sizeof(unsigned) * n_rows, st));
  argmax_rows_split_kernel<<<dim3(n_chunks, n_rows), 256, 0, st>>>(logits, vocab, chunk, tokens_out, sc);
  return check_launch("argmax_rows_split_kernel");
}
