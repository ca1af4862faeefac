// fitrig.cu -- C ABI (include/fitrig.h) of the B200-native FITrig hot path: context, launch
// logic, strip streaming.  All arithmetic of the method runs in the kernels of kernels.cuh; this
// file only allocates, encodes TMA descriptors, launches and copies.  There is no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <numeric>
#include <new>
#include <vector>

#include "fitrig.h"
#include "kernels.cuh"
#include "plan.h"

using namespace fitrig;

// ---------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(expr)                                                                               \
  do {                                                                                               \
    cudaError_t e__ = (expr);                                                                        \
    if (e__ != cudaSuccess) {                                                                        \
      const int code__ = (e__ == cudaErrorMemoryAllocation) ? FITRIG_ERR_NOMEM : FITRIG_ERR_CUDA;    \
      (void)cudaGetLastError();                                                                      \
      return fail(code__, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
    }                                                                                                \
  } while (0)

extern "C" const char* fitrig_last_error(void) { return g_err; }
extern "C" const char* fitrig_version(void) { return "fitrig-b200 0.1"; }

// ---------------------------------------------------------------------------------------------
// context
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static const int kMaxStripBuffers = 3;
static const int kPushSlots = 4;  // (a power of two: the kernels map ring slots with a mask)
// x_n, x_{n+1}, x_{n+2} of the unit being computed + the snapshot being copied
static const long long kHostStageCands = 4096;  // candidates fetched together with the count

struct CandHeader {
  unsigned long long total;
  unsigned long long pad;
};

struct DetectSlot {
  unsigned char* cand_dev;       // candidates (device list)
  long long cand_cap;
  unsigned char* cand_host;      // pinned + mapped: CandHeader + kHostStageCands candidates, written by the kernel
  unsigned char* cand_host_dev;  // device address of cand_host
  unsigned long long* counts_host;  // pinned + mapped: B per-stack totals
  unsigned long long* counts_host_dev;
  cudaEvent_t done;              // recorded behind the compaction kernel
  cudaStream_t stream;
  bool pending;
  long long cap, host_cap;       // of the launch in flight
};

struct TmapCache {  // the last TMA descriptor encoded (a resident stack is described by the same one call after call)
  bool valid = false;
  const float* base = nullptr;
  long long snap_stride = 0;
  int rows = 0, nslots = 0, box = 0, boxh = 0;
  CUtensorMap tm;
};

struct fitrig_ctx {
  NormParams prm;
  Tuning tune;         // FITRIG_* environment switches as they were when the context was created
  int H, W, L, U, Ty, Tx, B;
  long long nt, nmap;  // tiles per map row; B * U * nt
  int num_sms;
  long long max_pitch;
  fitrig_plan plan;
  EncodeTiledFn encode;
  TmapCache tmap;
  // map
  RawTile* raw;
  RawTile* raw_blocks;  // windows made of several cells (N_T = 32 * m, overlapping windows): one record per cell,
                        // merged into `raw` before the finalise
  CellGeom geo;         // cell edge, cells per window edge, cells between windows
  int Cy, Cx;           // cell grid
  int Ty32, Tx32;       // 32-pixel block grid of the fused kernel
  bool blocks_pending;  // the last tLISI launches wrote raw_blocks
  int cell_pix8;        // cells of one pixel: the tLISI kernels write 8-byte records (RawPix) ...
  int map_pix8;         // ... which are the map records themselves when a tile is one pixel
  float *q, *tlisi, *M_dev;
  unsigned* gmax_key;  // two sets of B order-preserving keys of the running global maxima, used by alternate calls:
  int key_idx;         // the finalise kernel of one call zeroes the keys of the next, so no memset sits in the stream
  bool keys_clean;
  StatPartial* parts;
  unsigned* counters;
  double *mu, *sigma;
  int fin_nblk, fin_grid, fin_chunk;
  int fin_user_row;    // -1: the caller's tLISI buffer receives the whole map; r >= 0: only map row r (real-time cube)
  // frequency branch
  float* eta;
  int* kstar;
  float* mag;  // [B][U/2][nt] magnitude spectrum
  double2* tw;
  StatPartial* sparts;
  unsigned* scounter;
  double *smu, *ssigma;
  int spec_nblk;
  bool eta_valid;
  // compaction: two result slots, so that the detection of one map can be fetched after the next map's work has
  // been queued (fitrig_detect_launch / fitrig_detect_fetch)
  DetectSlot slot[2];
  unsigned long long detect_launched, detect_fetched;
  unsigned long long* cstatus;
  unsigned* cticket;
  unsigned ticket_base;  // tickets drawn by all compaction launches so far (mod 2^32)
  unsigned compact_epoch;
  int compact_grid_max;
  // streaming
  float* strip_buf[kMaxStripBuffers];
  int n_strip_buf;
  long long strip_buf_elems;
  cudaStream_t copy_stream;
  cudaEvent_t ev_copied[kMaxStripBuffers], ev_free[kMaxStripBuffers], ev_entry;
  bool ev_free_pending[kMaxStripBuffers];
  // real-time mode (fitrig_push): ring of kPushSlots whole snapshots, running-maximum key, Fig. 14 timeline
  float* push_ring;
  unsigned* push_key;
  long long push_count;  // snapshots pushed so far
  long long push_next;   // next unit to compute
  cudaEvent_t ev_push_copied[4], ev_push_free[4];
  bool push_free_pending[4];
  // profiling
  bool profile;
  std::vector<cudaEvent_t> ev_pool;   // pairs: start, stop of each main-kernel launch since the last read
  int ev_used;
  std::vector<cudaEvent_t> fin_pool;  // pairs around each finalise launch since the last read
  int fin_used;
  std::vector<cudaEvent_t> tl_pool;   // fitrig_stream under profiling: per strip copy start / stop, kernel start / stop
  int tl_strips;                      // strips of the last profiled fitrig_stream
  bool have_map;
  long long launches;
  long long copies;  // host-to-device copy calls issued by fitrig_stream / fitrig_push
};

static void free_ctx(fitrig_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->prm.device);
  cudaDeviceSynchronize();
  cudaFree(c->raw); cudaFree(c->raw_blocks); cudaFree(c->q); cudaFree(c->tlisi); cudaFree(c->M_dev); cudaFree(c->gmax_key);
  cudaFree(c->parts); cudaFree(c->counters); cudaFree(c->mu); cudaFree(c->sigma);
  cudaFree(c->eta); cudaFree(c->kstar); cudaFree(c->mag); cudaFree(c->tw); cudaFree(c->sparts); cudaFree(c->scounter);
  cudaFree(c->smu); cudaFree(c->ssigma); cudaFree(c->cstatus); cudaFree(c->cticket);
  for (DetectSlot& d : c->slot) {
    cudaFree(d.cand_dev);
    if (d.cand_host) cudaFreeHost(d.cand_host);
    if (d.counts_host) cudaFreeHost(d.counts_host);
    if (d.done) cudaEventDestroy(d.done);
  }
  for (int i = 0; i < kMaxStripBuffers; ++i) {
    cudaFree(c->strip_buf[i]);
    if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
    if (c->ev_free[i]) cudaEventDestroy(c->ev_free[i]);
  }
  cudaFree(c->push_ring); cudaFree(c->push_key);
  for (int i = 0; i < kPushSlots; ++i) {
    if (c->ev_push_copied[i]) cudaEventDestroy(c->ev_push_copied[i]);
    if (c->ev_push_free[i]) cudaEventDestroy(c->ev_push_free[i]);
  }
  if (c->ev_entry) cudaEventDestroy(c->ev_entry);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  for (cudaEvent_t e : c->fin_pool) cudaEventDestroy(e);
  for (cudaEvent_t e : c->tl_pool) cudaEventDestroy(e);
  (void)cudaGetLastError();
  delete c;
}

template <int REF, bool ACC, int T>
static cudaError_t set_fused_attr_one() {
  return cudaFuncSetAttribute(tlisi_fused_kernel<REF, ACC, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemPerCta);
}

template <int REF>
static cudaError_t set_fused_attr() {
  cudaError_t e;
#define UNAL_ATTR(T)                                                                                                      \
  if ((e = cudaFuncSetAttribute(tlisi_fused_kernel<REF, false, T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                kMaxSmemPerCta)) != cudaSuccess) return e;
  UNAL_ATTR(32) UNAL_ATTR(16) UNAL_ATTR(8) UNAL_ATTR(4) UNAL_ATTR(2) UNAL_ATTR(1)
#undef UNAL_ATTR
  if ((e = set_fused_attr_one<REF, false, 32>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, true, 32>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, false, 16>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, true, 16>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, false, 8>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, true, 8>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, false, 4>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, true, 4>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, false, 2>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, true, 2>()) != cudaSuccess) return e;
  if ((e = set_fused_attr_one<REF, false, 1>()) != cudaSuccess) return e;
  return set_fused_attr_one<REF, true, 1>();
}

// The dynamic shared-memory limit of every tLISI kernel variant (also where the plan says generic: the unaligned variant
// and aligned strips of such a context ride the fused kernel).  A function attribute belongs to the device, not to a
// context: set once per device and process (with that device current), not on every fitrig_create.
static std::mutex g_attr_mu;
static bool g_attr_done[64];

static cudaError_t set_kernel_attributes_once(int device) {
  std::lock_guard<std::mutex> lock(g_attr_mu);
  if (device >= 0 && device < 64 && g_attr_done[device]) return cudaSuccess;
  cudaError_t e;
  if ((e = set_fused_attr<0>()) != cudaSuccess) return e;
  if ((e = set_fused_attr<1>()) != cudaSuccess) return e;
  if ((e = set_fused_attr<2>()) != cudaSuccess) return e;
#define MARCH_ATTR(R, S)                                                                                                    \
  if ((e = cudaFuncSetAttribute(tlisi_march_kernel<R, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemPerCta)) != \
      cudaSuccess) return e;
  MARCH_ATTR(0, false) MARCH_ATTR(1, false) MARCH_ATTR(2, false)
  MARCH_ATTR(0, true) MARCH_ATTR(1, true) MARCH_ATTR(2, true)
#undef MARCH_ATTR
  if (device >= 0 && device < 64) g_attr_done[device] = true;
  return cudaSuccess;
}

// A tLISI launch; with fp.dep != 0 as a programmatic dependent launch (the kernel places its own griddepcontrol.wait).
template <typename P>
static void launch_tlisi_kernel(void (*kernel)(const CUtensorMap, const P), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                const CUtensorMap& tm, const P& prm) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = prm.dep ? 1 : 0;
  (void)cudaLaunchKernelEx(&cfg, kernel, tm, prm);  // (the caller reads cudaGetLastError)
}

template <int REF, int T>
static void launch_fused_t(bool acc, dim3 grid, dim3 block, size_t smem, cudaStream_t st, const CUtensorMap& tm,
                           const FusedParams& fp) {
  if (acc) launch_tlisi_kernel(tlisi_fused_kernel<REF, true, T>, grid, block, smem, st, tm, fp);
  else launch_tlisi_kernel(tlisi_fused_kernel<REF, false, T>, grid, block, smem, st, tm, fp);
}

template <int REF>
static void launch_fused(bool acc, int tile, dim3 grid, dim3 block, size_t smem, cudaStream_t st, const CUtensorMap& tm,
                         const FusedParams& fp) {
  if (tile == 16) launch_fused_t<REF, 16>(acc, grid, block, smem, st, tm, fp);
  else if (tile == 8) launch_fused_t<REF, 8>(acc, grid, block, smem, st, tm, fp);
  else if (tile == 4) launch_fused_t<REF, 4>(acc, grid, block, smem, st, tm, fp);
  else if (tile == 2) launch_fused_t<REF, 2>(acc, grid, block, smem, st, tm, fp);
  else if (tile == 1) launch_fused_t<REF, 1>(acc, grid, block, smem, st, tm, fp);
  else launch_fused_t<REF, 32>(acc, grid, block, smem, st, tm, fp);
}

// A launch that may overlap its prologue with the tail of the previous kernel in the stream (programmatic dependent
// launch); every kernel launched this way starts with pdl_wait().
template <typename P>
static cudaError_t launch_chain(void (*kernel)(const P), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                const P& params) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, params);
}

extern "C" int fitrig_create(int32_t H, int32_t W, int32_t L, const fitrig_params* params, fitrig_ctx** out) {
  if (!out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_create: out is NULL");
  *out = nullptr;
  NormParams np;
  const char* why = "";
  int rc = normalize_params(H, W, L, params, &np, &why);
  if (rc != FITRIG_OK) return fail(rc, "fitrig_create: %s", why);

  int ndev = 0;
  CUDA_TRY(cudaGetDeviceCount(&ndev));
  if (np.device >= ndev) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_create: device %d of %d", np.device, ndev);
  CUDA_TRY(cudaSetDevice(np.device));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, np.device));
  if (prop.major < 10)
    return fail(FITRIG_ERR_CUDA, "fitrig_create: device %d is sm_%d%d; this library is built for sm_100a (B200) only",
                np.device, prop.major, prop.minor);

  fitrig_ctx* c = new (std::nothrow) fitrig_ctx();
  if (!c) return fail(FITRIG_ERR_NOMEM, "fitrig_create: host allocation failed");
  c->prm = np;
  c->tune = read_tuning_env();
  c->H = H; c->W = W; c->L = L; c->U = L / np.accumulate - 2; c->B = np.batch;
  c->num_sms = prop.multiProcessorCount;
  c->max_pitch = (long long)prop.memPitch;
  rc = fitrig_plan_query(H, W, L, params, c->num_sms, &c->plan);
  if (rc != FITRIG_OK) { delete c; return fail(rc, "fitrig_create: plan failed"); }
  c->Ty = c->plan.Ty; c->Tx = c->plan.Tx;
  c->nt = (long long)c->Ty * c->Tx;
  c->nmap = c->nt * c->U * c->B;
  if (c->nmap > 0x7fffffffll || c->nt > 0x7fffffffll) {
    delete c;
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_create: map of %lld entries is too large", c->nmap);
  }
  const long long R = (long long)c->B * c->U;  // map rows

#define CTX_TRY(expr)                                                                                 \
  do {                                                                                                \
    cudaError_t e__ = (expr);                                                                         \
    if (e__ != cudaSuccess) {                                                                         \
      const int code__ = (e__ == cudaErrorMemoryAllocation) ? FITRIG_ERR_NOMEM : FITRIG_ERR_CUDA;     \
      (void)cudaGetLastError();                                                                       \
      free_ctx(c);                                                                                    \
      return fail(code__, "fitrig_create: %s failed: %s", #expr, cudaGetErrorString(e__));            \
    }                                                                                                 \
  } while (0)

  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  CTX_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
  if (!fn || qres != cudaDriverEntryPointSuccess) {
    free_ctx(c);
    return fail(FITRIG_ERR_CUDA, "fitrig_create: cuTensorMapEncodeTiled not available in this driver");
  }
  c->encode = (EncodeTiledFn)fn;

  CTX_TRY(cudaMalloc(&c->raw, sizeof(RawTile) * c->nmap));
  c->Ty32 = (H + kFastTile - 1) / kFastTile; c->Tx32 = (W + kFastTile - 1) / kFastTile;
  c->geo = cell_geom(np.tile, np.stride);
  c->cell_pix8 = c->geo.cell == 1;
  c->map_pix8 = c->cell_pix8 && c->geo.m == 1;
  c->Cy = (H + c->geo.cell - 1) / c->geo.cell; c->Cx = (W + c->geo.cell - 1) / c->geo.cell;
  if (c->geo.m > 1) CTX_TRY(cudaMalloc(&c->raw_blocks, sizeof(RawTile) * (size_t)R * c->Cy * c->Cx));
  CTX_TRY(cudaMalloc(&c->q, sizeof(float) * c->nmap));
  CTX_TRY(cudaMalloc(&c->tlisi, sizeof(float) * c->nmap));
  CTX_TRY(cudaMalloc(&c->M_dev, sizeof(float) * c->B));
  CTX_TRY(cudaMalloc(&c->gmax_key, 2 * sizeof(unsigned) * c->B));
  CTX_TRY(cudaMemset(c->gmax_key, 0, 2 * sizeof(unsigned) * c->B));
  c->keys_clean = true;
  // map entries per block and pass: every chunk costs a block-wide reduction and a hand-over (fence + atomic), so big
  // maps (small tiles) get chunks large enough that each block of the grid sees only a few of them
  const long long fin_blocks = 8ll * c->num_sms;
  c->fin_chunk = (int)std::min<long long>(kFinChunkMax, std::max<long long>(kFinChunk, (c->nmap / (2 * fin_blocks) + 255) / 256 * 256));
  c->fin_nblk = (int)((c->nt + c->fin_chunk - 1) / c->fin_chunk);
  c->fin_grid = (int)std::max<long long>(1, std::min<long long>(R * c->fin_nblk, fin_blocks));
  c->fin_user_row = -1;
  CTX_TRY(cudaMalloc(&c->parts, sizeof(StatPartial) * R * c->fin_nblk));
  CTX_TRY(cudaMalloc(&c->counters, sizeof(unsigned) * R));
  CTX_TRY(cudaMemset(c->counters, 0, sizeof(unsigned) * R));
  CTX_TRY(cudaMalloc(&c->mu, sizeof(double) * R));
  CTX_TRY(cudaMalloc(&c->sigma, sizeof(double) * R));
  if (np.branch == FITRIG_BRANCH_FREQUENCY) {
    CTX_TRY(cudaMalloc(&c->eta, sizeof(float) * c->nt * c->B));
    CTX_TRY(cudaMalloc(&c->kstar, sizeof(int) * c->nt * c->B));
    CTX_TRY(cudaMalloc(&c->mag, sizeof(float) * (size_t)std::max(1, c->U / 2) * c->nt * c->B));
    CTX_TRY(cudaMalloc(&c->tw, sizeof(double2) * c->U));
    std::vector<double2> tw(c->U);
    for (int j = 0; j < c->U; ++j) {  // exp(-2 pi i j / U), Eq. 10's Fourier kernel (R17)
      const double a = -2.0 * M_PI * (double)j / (double)c->U;
      tw[j].x = cos(a);
      tw[j].y = sin(a);
    }
    CTX_TRY(cudaMemcpy(c->tw, tw.data(), sizeof(double2) * c->U, cudaMemcpyHostToDevice));
    if (sizeof(double2) * c->U > 48 * 1024)
      CTX_TRY(cudaFuncSetAttribute(dft_mag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double2) * c->U)));
    c->spec_nblk = (int)((c->nt + kSpecChunk - 1) / kSpecChunk);
    CTX_TRY(cudaMalloc(&c->sparts, sizeof(StatPartial) * c->spec_nblk * c->B));
    CTX_TRY(cudaMalloc(&c->scounter, sizeof(unsigned) * c->B));
    CTX_TRY(cudaMemset(c->scounter, 0, sizeof(unsigned) * c->B));
    CTX_TRY(cudaMalloc(&c->smu, sizeof(double) * c->B));
    CTX_TRY(cudaMalloc(&c->ssigma, sizeof(double) * c->B));
  }
  int occ = 0;
  CTX_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, compact_kernel, 512, 0));
  c->compact_grid_max = std::max(1, occ) * c->num_sms;
  CTX_TRY(cudaMalloc(&c->cticket, sizeof(unsigned)));
  CTX_TRY(cudaMemset(c->cticket, 0, sizeof(unsigned)));
  c->ticket_base = 0;
  CTX_TRY(cudaMalloc(&c->cstatus, sizeof(unsigned long long) * c->compact_grid_max));
  CTX_TRY(cudaMemset(c->cstatus, 0, sizeof(unsigned long long) * c->compact_grid_max));
  c->compact_epoch = 0;
  for (DetectSlot& d : c->slot) {
    d.cand_cap = kHostStageCands;
    CTX_TRY(cudaMalloc(&d.cand_dev, sizeof(fitrig_candidate) * d.cand_cap));
    CTX_TRY(cudaHostAlloc(&d.cand_host, sizeof(CandHeader) + sizeof(fitrig_candidate) * kHostStageCands,
                          cudaHostAllocMapped));
    CTX_TRY(cudaHostGetDevicePointer((void**)&d.cand_host_dev, d.cand_host, 0));
    CTX_TRY(cudaHostAlloc(&d.counts_host, sizeof(unsigned long long) * c->B, cudaHostAllocMapped));
    CTX_TRY(cudaHostGetDevicePointer((void**)&d.counts_host_dev, d.counts_host, 0));
    CTX_TRY(cudaEventCreateWithFlags(&d.done, cudaEventDisableTiming));
  }
  CTX_TRY(set_kernel_attributes_once(c->prm.device));
#undef CTX_TRY
  *out = c;
  return FITRIG_OK;
}

extern "C" int fitrig_destroy(fitrig_ctx* ctx) {
  free_ctx(ctx);
  return FITRIG_OK;
}

extern "C" int fitrig_map_dims(const fitrig_ctx* ctx, int32_t* units, int32_t* Ty, int32_t* Tx) {
  if (!ctx) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_map_dims: ctx is NULL");
  if (units) *units = ctx->U;
  if (Ty) *Ty = ctx->Ty;
  if (Tx) *Tx = ctx->Tx;
  return FITRIG_OK;
}

// ---------------------------------------------------------------------------------------------
// launches
// ---------------------------------------------------------------------------------------------
static int prof_begin(fitrig_ctx* c, cudaStream_t st) {
  if (!c->profile) return FITRIG_OK;
  while ((int)c->ev_pool.size() < 2 * (c->ev_used + 1)) {
    cudaEvent_t e;
    CUDA_TRY(cudaEventCreate(&e));
    c->ev_pool.push_back(e);
  }
  CUDA_TRY(cudaEventRecord(c->ev_pool[2 * c->ev_used], st));
  return FITRIG_OK;
}
static int prof_end(fitrig_ctx* c, cudaStream_t st) {
  if (!c->profile) return FITRIG_OK;
  CUDA_TRY(cudaEventRecord(c->ev_pool[2 * c->ev_used + 1], st));
  c->ev_used++;
  return FITRIG_OK;
}

// The TMA descriptor of `nslots` images of rows x W (rows `snap_stride` elements apart per image) with boxes of
// box x boxh pixels; the last one encoded is kept (a resident stack is described by the same one call after call).
static int get_tmap(fitrig_ctx* c, const float* base, long long snap_stride, int rows, int nslots, int box, int boxh,
                    const CUtensorMap** out) {
  TmapCache& tc = c->tmap;
  if (!(tc.valid && tc.base == base && tc.snap_stride == snap_stride && tc.rows == rows && tc.nslots == nslots &&
        tc.box == box && tc.boxh == boxh)) {
    const cuuint64_t gdim[3] = {(cuuint64_t)c->W, (cuuint64_t)rows, (cuuint64_t)nslots};
    const cuuint64_t gstr[2] = {(cuuint64_t)c->W * 4, (cuuint64_t)snap_stride * 4};
    const cuuint32_t bx[3] = {(cuuint32_t)box, (cuuint32_t)boxh, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = c->encode(&tc.tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base, gdim, gstr, bx, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { tc.valid = false; return fail(FITRIG_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r); }
    tc.valid = true; tc.base = base; tc.snap_stride = snap_stride; tc.rows = rows; tc.nslots = nslots; tc.box = box; tc.boxh = boxh;
  }
  *out = &tc.tm;
  return FITRIG_OK;
}

// tLISI partial sums of `rows` image rows (all L snapshots) that start at tile row ty_base.
// base: device pointer to snapshot 0 of those rows; snap_stride: elements between snapshots.
struct RowsOpt {
  int z0 = 0, zmod = 0;     // real-time ring: snapshot s of the launch is slot (z0 + s) % zmod of `base`
  unsigned* key = nullptr;  // global-maximum key to fold into (default: the key of stack `stack` of the current call)
  int stack = 0;            // batch entry: the records go to map rows stack * U ..
  int units = 0;            // units computed by this launch (0: all U of the context)
  int row0 = 0;             // ... starting at this row of the stack's U rows (the real-time cube's ring slot)
  int dep = 0;              // programmatic dependent launch of the tLISI kernel (FusedParams::dep)
};

static int launch_tlisi_rows(fitrig_ctx* c, const float* base, long long snap_stride, int rows, int r0,
                             bool with_max, cudaStream_t st, const RowsOpt& opt = RowsOpt()) {
  const int tile = c->geo.cell;        // what the kernels reduce: cells (the tile itself in the plain case)
  const int ty_base = r0 / tile;       // first cell row of this launch
  const bool cells = c->geo.m > 1;     // records go to raw_blocks and are merged into windows before the finalise
  const int out_Ty = cells ? c->Cy : c->Ty, out_Tx = cells ? c->Cx : c->Tx;
  const long long first_row = (long long)opt.stack * c->U + opt.row0;
  // (cells of one pixel are 8-byte RawPix records, which the kernels index from this base: the offset is in records of that size)
  const size_t rec_bytes = c->cell_pix8 ? sizeof(RawPix) : sizeof(RawTile);
  RawTile* const out_raw = reinterpret_cast<RawTile*>(reinterpret_cast<unsigned char*>(cells ? c->raw_blocks : c->raw) +
                                                      (size_t)(first_row * out_Ty * out_Tx) * rec_bytes);
  const int units = opt.units ? opt.units : c->U;
  unsigned* key = opt.key ? opt.key : c->gmax_key + c->key_idx * c->B + opt.stack;
  const int nslots = opt.zmod ? opt.zmod : c->L;
  const int rows_tiles = (rows + tile - 1) / tile;
  fitrig_plan pl = c->plan;
  const bool aligned = ((uintptr_t)base % 16 == 0) && (snap_stride % 4 == 0) && (c->W % 4 == 0);  // what TMA needs
  // Rows that do not start on 16-byte boundaries: cells of 32 pixels of ONE contiguous stack still ride the fused kernel,
  // through a tensor map of "super rows" of k image rows (kernels.cuh, UNAL); everything else takes the generic kernel.
  bool unal = false;
  int unal_k = 1;
  CUtensorMap tm_unal;
  const int unal_a = (int)(((uintptr_t)base >> 2) & 3);
  if (!aligned && tile <= kFastTile && fused_tile(tile) && c->prm.accumulate == 1 && !c->tune.force_generic && !c->tune.no_unaligned_fused &&
      (uintptr_t)base % 4 == 0 && snap_stride % c->W == 0 && snap_stride / c->W >= rows && r0 % kFastTile == 0) {
    unal_k = 4 / std::gcd(c->W, 4);
    // (dim0 = k W + a_off exceeds the row stride of k W by a_off: rows of the tensor map overlap, which the driver accepts
    // and which reads the flat continuation -- checked on the B200)
    unal = (nslots * (snap_stride / c->W)) % unal_k == 0 && (long long)unal_k * c->W + 4 <= 0x7fffffffll &&
           nslots * (snap_stride / c->W) <= 0x7fffffffll;
    if (unal) {
      Tuning tn = c->tune;
      plan_launch_fused(tile, c->W, rows, units, c->num_sms, tn, /*extra_row_bytes=*/16, &pl);
      // super rows of k image rows, from the 16-byte boundary at or below the base.  Rows of this map overlap (dim0 exceeds
      // the row stride), which the B200's driver accepts; a driver that refuses it sends the image to the generic kernel
      const cuuint64_t gdim[2] = {(cuuint64_t)unal_k * c->W + unal_a, (cuuint64_t)(nslots * (snap_stride / c->W) / unal_k)};
      const cuuint64_t gstr[1] = {(cuuint64_t)unal_k * c->W * 4};
      const cuuint32_t bx[2] = {(cuuint32_t)(pl.box_tiles * kFastTile + 4), (cuuint32_t)(kFastTile / unal_k)};
      const cuuint32_t estr[2] = {1, 1};
      CUresult r = c->tune.fail_unaligned_encode
                       ? CUDA_ERROR_INVALID_VALUE
                       : c->encode(&tm_unal, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)(base - unal_a), gdim, gstr, bx, estr,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) {
        unal = false;
        pl = c->plan;
      }
    }
  }
  if (pl.path == 0 && !aligned && !unal) pl.path = 1;  // TMA needs 16-byte aligned base and strides
  if (pl.path == 0 && r0 % kFastTile != 0) pl.path = 1;  // strips must start on a 32-row block
  if (pl.path == 0 && !unal && (rows != c->H || units != c->U)) plan_launch(tile, c->W, rows, units, c->num_sms, c->tune, &pl);

  // generic path: the time-marching kernel (TMA boxes where the image allows, else cp.async copies into shifted rows)
  MarchPlan mp = MarchPlan();
  bool tma = false;
  if (pl.path != 0 && c->prm.accumulate == 1 && !c->tune.old_generic) {
    mp = plan_march(tile, c->W, rows, units, c->num_sms, c->tune, false);
    tma = mp.ok && aligned && mp.x_aligned;
    if (mp.ok && !tma) mp = plan_march(tile, c->W, rows, units, c->num_sms, c->tune, true);
  }
  int rc = prof_begin(c, st);
  if (rc) return rc;
  if (pl.path == 0) {
    const CUtensorMap* tmp = nullptr;
    if (unal) {
      tmp = &tm_unal;
    } else {
      rc = get_tmap(c, base, snap_stride, rows, nslots, pl.box_tiles * kFastTile, kFastTile, &tmp);
      if (rc) return rc;
    }
    const CUtensorMap& tm = *tmp;
    FusedParams fp;
    fp.k_rows = unal_k; fp.a_off = unal_a; fp.rows = rows; fp.srows = (int)(snap_stride / c->W); fp.even_shifts = (c->W % 2 == 0) && (unal_a % 2 == 0);
    fp.raw = out_raw; fp.gmax_key = key;
    fp.z0 = opt.z0; fp.zmask = opt.zmod ? opt.zmod - 1 : 0x7fffffff; fp.acc = c->prm.accumulate;
    fp.base = base; fp.snap_stride = snap_stride; fp.W = c->W;
    fp.Tx = out_Tx; fp.Ty = out_Ty; fp.Tx32 = c->Tx32;
    fp.rows_tiles = (rows + kFastTile - 1) / kFastTile; fp.ty_base = ty_base;
    fp.ty_end = std::min(out_Ty, ty_base + rows_tiles);
    fp.U = units;
    fp.ntw = pl.box_tiles; fp.ngx = (fp.Tx32 + pl.box_tiles - 1) / pl.box_tiles; fp.nstage = pl.stages;
    const long long G = (long long)fp.rows_tiles * fp.ngx * units;
    if (G > 0x7fffffffll) return fail(FITRIG_ERR_INVALID_ARG, "fused path: too many (box, unit) pairs for one launch");
    fp.G = (int)G;
    fp.evict_first = c->tune.evict_first;
    fp.C = c->prm.C;
    fp.dep = (c->tune.no_pdl || c->profile) ? 0 : opt.dep;
    const dim3 grid(pl.grid), block(32 * pl.warps_per_cta);
    if (unal) {
#define UNAL_LAUNCH(R, T) launch_tlisi_kernel(tlisi_fused_kernel<R, false, T, true>, grid, block, (size_t)pl.smem_bytes, st, tm, fp)
#define UNAL_TILES(R)                                                                                               \
  (tile == 16 ? UNAL_LAUNCH(R, 16) : tile == 8 ? UNAL_LAUNCH(R, 8) : tile == 4 ? UNAL_LAUNCH(R, 4) : tile == 2 ? UNAL_LAUNCH(R, 2) \
   : tile == 1 ? UNAL_LAUNCH(R, 1) : UNAL_LAUNCH(R, 32))
      switch (c->prm.ref_mode) {
        case FITRIG_REF_ABS: UNAL_TILES(FITRIG_REF_ABS); break;
        case FITRIG_REF_LITERAL: UNAL_TILES(FITRIG_REF_LITERAL); break;
        default: UNAL_TILES(FITRIG_REF_FLOOR); break;
      }
#undef UNAL_TILES
#undef UNAL_LAUNCH
    } else
    switch (c->prm.ref_mode) {
      case FITRIG_REF_ABS: launch_fused<FITRIG_REF_ABS>(fp.acc > 1, tile, grid, block, pl.smem_bytes, st, tm, fp); break;
      case FITRIG_REF_LITERAL: launch_fused<FITRIG_REF_LITERAL>(fp.acc > 1, tile, grid, block, pl.smem_bytes, st, tm, fp); break;
      default: launch_fused<FITRIG_REF_FLOOR>(fp.acc > 1, tile, grid, block, pl.smem_bytes, st, tm, fp); break;
    }
    CUDA_TRY(cudaGetLastError());
    c->launches++;
    if (cells) c->blocks_pending = true;
  } else if (mp.ok) {
    // any cell size / width / alignment, every snapshot byte read once (time-marching through a shared-memory ring)
    const CUtensorMap* tmp = &c->tmap.tm;  // (unused by the cp.async variant)
    if (tma) {
      rc = get_tmap(c, base, snap_stride, rows, nslots, mp.bwp, mp.bh, &tmp);
      if (rc) return rc;
    }
    MarchParams q;
    q.raw = out_raw; q.gmax_key = key; q.base = base; q.snap_stride = snap_stride; q.W = c->W; q.rows = rows;
    q.Tx = out_Tx; q.Ty = out_Ty; q.ty_base = ty_base; q.ty_end = std::min(out_Ty, ty_base + rows_tiles);
    q.U = units; q.c = tile; q.ntx = mp.ntx; q.nty = mp.nty; q.bwp = mp.bwp; q.bh = mp.bh; q.pitch = mp.pitch; q.ngx = mp.ngx;
    q.nstage = mp.nstage; q.G = (int)((long long)mp.ngx * mp.ngy * units);
    q.z0 = opt.z0; q.zmask = opt.zmod ? opt.zmod - 1 : 0x7fffffff; q.tma = tma ? 1 : 0; q.C = c->prm.C;
    q.ncons = mp.ncons; q.nprod = mp.nprod;
    q.dep = (c->tune.no_pdl || c->profile) ? 0 : opt.dep;
    q.pix8 = c->cell_pix8;
    const dim3 grid(mp.grid), block(32 * (q.ncons + q.nprod));
    auto launch = [&](auto kernel) { launch_tlisi_kernel(kernel, grid, block, (size_t)mp.smem_bytes, st, *tmp, q); };
#define MARCH_LAUNCH(R) (tma ? launch(tlisi_march_kernel<R, false>) : launch(tlisi_march_kernel<R, true>))
    switch (c->prm.ref_mode) {
      case FITRIG_REF_ABS: MARCH_LAUNCH(FITRIG_REF_ABS); break;
      case FITRIG_REF_LITERAL: MARCH_LAUNCH(FITRIG_REF_LITERAL); break;
      default: MARCH_LAUNCH(FITRIG_REF_FLOOR); break;
    }
#undef MARCH_LAUNCH
    CUDA_TRY(cudaGetLastError());
    c->launches++;
    if (cells) c->blocks_pending = true;
  } else {
    if (with_max) {
      // rows of each snapshot are contiguous (full width), so one launch per snapshot covers them
      const int g = c->prm.accumulate;
      for (int s = 0; s < units + 2; ++s) {  // (accumulated) images; the ring mode never accumulates
        const int slot = opt.zmod ? (opt.z0 + s) % opt.zmod : s * g;
        stack_max_kernel<<<std::min(4 * c->num_sms, 1024), 256, 0, st>>>(base + (long long)slot * snap_stride,
                                                                       (long long)rows * c->W, g, snap_stride, key);
        CUDA_TRY(cudaGetLastError());
        c->launches++;
      }
    }
    GenericParams gp;
    gp.base = base; gp.snap_stride = snap_stride; gp.rows = rows; gp.W = c->W; gp.tile = tile;
    gp.raw = out_raw; gp.Tx = out_Tx; gp.Ty = out_Ty; gp.ty_base = ty_base; gp.rows_tiles = rows_tiles; gp.U = units;
    if (cells) c->blocks_pending = true;
    int G = 1;
    const long long n_t = (long long)tile * tile;
    while (G < 32 && G < n_t) G <<= 1;
    gp.G = G;
    gp.z0 = opt.z0; gp.zmask = opt.zmod ? opt.zmod - 1 : 0x7fffffff; gp.acc = c->prm.accumulate;
    gp.C = c->prm.C;
    gp.pix8 = c->cell_pix8;
    const long long groups = (long long)rows_tiles * out_Tx * units;
    const long long threads = groups * G;
    const long long blocks = (threads + 255) / 256;
    if (blocks > 0x7fffffffll) return fail(FITRIG_ERR_INVALID_ARG, "generic path: too many tiles for one launch");
    switch (c->prm.ref_mode) {
      case FITRIG_REF_ABS: tlisi_generic_kernel<FITRIG_REF_ABS><<<(unsigned)blocks, 256, 0, st>>>(gp); break;
      case FITRIG_REF_LITERAL: tlisi_generic_kernel<FITRIG_REF_LITERAL><<<(unsigned)blocks, 256, 0, st>>>(gp); break;
      default: tlisi_generic_kernel<FITRIG_REF_FLOOR><<<(unsigned)blocks, 256, 0, st>>>(gp); break;
    }
    CUDA_TRY(cudaGetLastError());
    c->launches++;
  }
  return prof_end(c, st);
}

static void fill_finalize_params(fitrig_ctx* c, FinalizeParams* fp, float* d_tlisi_user, const unsigned* keys) {
  fp->raw = c->raw; fp->q = c->q; fp->tlisi = c->tlisi; fp->tlisi_user = d_tlisi_user;
  fp->gmax_key = keys; fp->gmax_key_next = c->gmax_key + (c->key_idx ^ 1) * c->B;
  fp->M_out = c->M_dev; fp->M_override = c->prm.M_override; fp->C = c->prm.C;
  fp->H = c->H; fp->W = c->W; fp->tile = c->prm.tile; fp->stride = c->prm.stride; fp->Ty = c->Ty; fp->Tx = c->Tx;
  fp->U = c->U; fp->B = c->B;
  fp->nblk = c->fin_nblk; fp->chunk = c->fin_chunk; fp->parts = c->parts; fp->counters = c->counters; fp->mu = c->mu; fp->sigma = c->sigma;
  fp->shard_all = nullptr; fp->shard_world = 0;
  fp->user_row = c->fin_user_row;
  fp->pix8 = c->map_pix8;
}

// keys: one global-maximum key per stack (default: the keys of the current call)
static int launch_finalize(fitrig_ctx* c, float* d_tlisi_user, cudaStream_t st, unsigned* keys = nullptr) {
  bool chained = !c->tune.no_pdl && !c->profile;  // behind the tLISI kernel (an event record in between breaks the chain)
  if (c->raw_blocks && c->blocks_pending) {  // cell records -> window records
    MergeParams mp;
    mp.cells = c->raw_blocks; mp.raw = c->raw; mp.U = c->U * c->B; mp.Ty = c->Ty; mp.Tx = c->Tx;
    mp.Cy = c->Cy; mp.Cx = c->Cx; mp.m = c->geo.m; mp.step = c->geo.step; mp.cell = c->geo.cell; mp.tile = c->prm.tile;
    mp.pix8 = c->cell_pix8;
    const long long n = c->nmap * (mp.m * mp.m >= 32 ? 32 : 1);  // threads wanted (a warp per window of many cells)
    merge_cells_kernel<<<(unsigned)std::min<long long>((n + 255) / 256, 16 * c->num_sms), 256, 0, st>>>(mp);
    CUDA_TRY(cudaGetLastError());
    c->launches++;
    c->blocks_pending = false;
  }
  FinalizeParams fp;
  fill_finalize_params(c, &fp, d_tlisi_user, keys ? keys : c->gmax_key + c->key_idx * c->B);
  if (c->profile) {
    while ((int)c->fin_pool.size() < 2 * (c->fin_used + 1)) {
      cudaEvent_t e;
      CUDA_TRY(cudaEventCreate(&e));
      c->fin_pool.push_back(e);
    }
    CUDA_TRY(cudaEventRecord(c->fin_pool[2 * c->fin_used], st));
  }
  CUDA_TRY(launch_chain(c->map_pix8 ? finalize_kernel<true> : finalize_kernel<false>, dim3(c->fin_grid), dim3(256), 0, st, chained, fp));
  if (c->profile) { CUDA_TRY(cudaEventRecord(c->fin_pool[2 * c->fin_used + 1], st)); c->fin_used++; }
  c->launches++;
  c->have_map = true;
  c->eta_valid = false;
  c->keys_clean = true;
  return FITRIG_OK;
}

static int begin_call(fitrig_ctx* c, cudaStream_t st) {
  CUDA_TRY(cudaSetDevice(c->prm.device));
  if (!c->keys_clean) CUDA_TRY(cudaMemsetAsync(c->gmax_key, 0, 2 * sizeof(unsigned) * c->B, st));  // a call failed half way
  c->keys_clean = false;
  c->key_idx ^= 1;
  return FITRIG_OK;
}

extern "C" int fitrig_tlisi_batch(fitrig_ctx* c, const float* const* d_stacks, float* d_tlisi, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_tlisi_batch: ctx is NULL");
  if (!d_stacks) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_tlisi_batch: d_stacks is NULL");
  for (int b = 0; b < c->B; ++b)
    if (!d_stacks[b]) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_tlisi_batch: d_stacks[%d] is NULL", b);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = begin_call(c, st);
  if (rc) return rc;
  for (int b = 0; b < c->B; ++b) {
    RowsOpt opt;
    opt.stack = b;
    opt.dep = b == 0 ? 1 : 2;  // the stacks are independent: their kernels overlap tail and ramp-up
    rc = launch_tlisi_rows(c, d_stacks[b], (long long)c->H * c->W, c->H, 0, true, st, opt);
    if (rc) return rc;
  }
  return launch_finalize(c, d_tlisi, st);
}

extern "C" int fitrig_tlisi(fitrig_ctx* c, const float* d_stack, float* d_tlisi, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_tlisi: ctx is NULL");
  if (!d_stack) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_tlisi: d_stack is NULL");
  std::vector<const float*> ptrs(c->B);
  for (int b = 0; b < c->B; ++b) ptrs[b] = d_stack + (size_t)b * c->L * c->H * c->W;
  return fitrig_tlisi_batch(c, ptrs.data(), d_tlisi, cuda_stream);
}

// fitrig_stream's strip loop; on an error the caller drains the copy stream
static int stream_strips(fitrig_ctx* c, const float* const* h_snapshots, cudaStream_t st) {
  const int rows_per = c->plan.strip_rows, nstrips = c->plan.n_strips, nbuf = c->plan.n_strip_buffers;
  const long long snap_stride = (long long)rows_per * c->W;
  // snapshots that sit at a constant distance in host memory (one [L][H][W] allocation, the usual case) let a
  // strip travel as one pitched copy instead of L small ones; pitches are limited to cudaDeviceProp::memPitch
  long long host_stride = h_snapshots[1] - h_snapshots[0];
  bool pitched = host_stride >= (long long)c->H * c->W && host_stride * 4 <= c->max_pitch && snap_stride * 4 <= c->max_pitch &&
                 c->tune.no_pitched_copy == 0;
  for (int s = 2; s < c->L && pitched; ++s) pitched = (h_snapshots[s] - h_snapshots[s - 1]) == host_stride;
  c->tl_strips = 0;
  if (c->profile) {  // the copy / kernel timeline of this call (fitrig_stream_timeline)
    while ((int)c->tl_pool.size() < 4 * nstrips) {
      cudaEvent_t e;
      CUDA_TRY(cudaEventCreate(&e));
      c->tl_pool.push_back(e);
    }
  }
  for (int i = 0; i < nstrips; ++i) {
    const int b = i % nbuf;
    const int r0 = i * rows_per;
    const int rows = std::min(rows_per, c->H - r0);
    if (c->ev_free_pending[b]) CUDA_TRY(cudaStreamWaitEvent(c->copy_stream, c->ev_free[b], 0));
    if (c->profile) CUDA_TRY(cudaEventRecord(c->tl_pool[4 * i], c->copy_stream));
    if (pitched) {  // equally spaced snapshots: the whole strip (L row blocks) is ONE pitched copy
      cudaError_t e2 = cudaMemcpy2DAsync(c->strip_buf[b], sizeof(float) * snap_stride, h_snapshots[0] + (long long)r0 * c->W,
                                         sizeof(float) * host_stride, sizeof(float) * (long long)rows * c->W, c->L,
                                         cudaMemcpyHostToDevice, c->copy_stream);
      if (e2 == cudaErrorInvalidValue) {  // equally spaced but separate allocations: the range check refuses
        (void)cudaGetLastError();
        pitched = false;
      } else {
        CUDA_TRY(e2);
        c->copies++;
      }
    }
    if (!pitched) {
      for (int s = 0; s < c->L; ++s) {  // snapshot s, rows r0..r0+rows: contiguous on both sides
        CUDA_TRY(cudaMemcpyAsync(c->strip_buf[b] + (long long)s * snap_stride, h_snapshots[s] + (long long)r0 * c->W,
                                 sizeof(float) * (long long)rows * c->W, cudaMemcpyHostToDevice, c->copy_stream));
        c->copies++;
      }
    }
    if (c->profile) CUDA_TRY(cudaEventRecord(c->tl_pool[4 * i + 1], c->copy_stream));
    CUDA_TRY(cudaEventRecord(c->ev_copied[b], c->copy_stream));
    CUDA_TRY(cudaStreamWaitEvent(st, c->ev_copied[b], 0));
    if (c->profile) CUDA_TRY(cudaEventRecord(c->tl_pool[4 * i + 2], st));
    int rc = launch_tlisi_rows(c, c->strip_buf[b], snap_stride, rows, r0, true, st);
    if (rc) return rc;
    if (c->profile) CUDA_TRY(cudaEventRecord(c->tl_pool[4 * i + 3], st));
    CUDA_TRY(cudaEventRecord(c->ev_free[b], st));
    c->ev_free_pending[b] = true;
  }
  if (c->profile) c->tl_strips = nstrips;
  return FITRIG_OK;
}

extern "C" int fitrig_stream(fitrig_ctx* c, const float* const* h_snapshots, float* h_tlisi, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream: ctx is NULL");
  if (!h_snapshots) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream: h_snapshots is NULL");
  if (c->B != 1) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream: not with params.batch > 1");
  for (int s = 0; s < c->L; ++s)
    if (!h_snapshots[s]) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream: h_snapshots[%d] is NULL", s);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  const int rows_per = c->plan.strip_rows, nbuf = c->plan.n_strip_buffers;
  if (!c->copy_stream) CUDA_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
  if (!c->ev_entry) CUDA_TRY(cudaEventCreateWithFlags(&c->ev_entry, cudaEventDisableTiming));
  if (!c->n_strip_buf) {
    c->strip_buf_elems = (long long)c->L * rows_per * c->W;
    for (int b = 0; b < nbuf; ++b) {
      CUDA_TRY(cudaMalloc(&c->strip_buf[b], sizeof(float) * c->strip_buf_elems));
      CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copied[b], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&c->ev_free[b], cudaEventDisableTiming));
    }
    c->n_strip_buf = nbuf;
  }
  int rc = begin_call(c, st);
  if (rc) return rc;
  // the copy stream may not run ahead of work already queued on the caller's stream
  CUDA_TRY(cudaEventRecord(c->ev_entry, st));
  CUDA_TRY(cudaStreamWaitEvent(c->copy_stream, c->ev_entry, 0));
  for (int b = 0; b < nbuf; ++b) c->ev_free_pending[b] = false;
  rc = stream_strips(c, h_snapshots, st);
  if (rc == FITRIG_OK) rc = launch_finalize(c, nullptr, st);
  if (rc != FITRIG_OK) {
    // leave nothing queued behind a failed call: the copies still in flight read the caller's buffers and write the
    // strip buffers the next call will reuse (the message of the original failure is kept)
    (void)cudaStreamSynchronize(c->copy_stream);
    (void)cudaStreamSynchronize(st);
    (void)cudaGetLastError();
    for (int b = 0; b < nbuf; ++b) c->ev_free_pending[b] = false;
    c->have_map = false;
    return rc;
  }
  if (h_tlisi) CUDA_TRY(cudaMemcpyAsync(h_tlisi, c->tlisi, sizeof(float) * c->nmap, cudaMemcpyDeviceToHost, st));
  return FITRIG_OK;
}

static int detect_launch_core(fitrig_ctx* c, float tau, int64_t capacity, void* cuda_stream, int unit_offset);
static int detect_fetch_core(fitrig_ctx* c, fitrig_candidate* h_out, int64_t* n_found, int64_t* n_per_stack);

static int detect_core(fitrig_ctx* c, float tau, fitrig_candidate* h_out, int64_t capacity, int64_t* n_found,
                       int64_t* n_per_stack, void* cuda_stream, int unit_offset) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect: ctx is NULL");
  if (!n_found) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect: n_found is NULL");
  if (capacity < 0 || (capacity > 0 && !h_out)) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect: bad h_out/capacity");
  if (c->detect_launched != c->detect_fetched)
    return fail(FITRIG_ERR_STATE, "fitrig_detect: a fitrig_detect_launch has not been fetched yet");
  int rc = detect_launch_core(c, tau, capacity, cuda_stream, unit_offset);
  if (rc) return rc;
  return detect_fetch_core(c, h_out, n_found, n_per_stack);
}

extern "C" int fitrig_detect(fitrig_ctx* c, float tau, fitrig_candidate* h_out, int64_t capacity, int64_t* n_found,
                             void* cuda_stream) {
  return detect_core(c, tau, h_out, capacity, n_found, nullptr, cuda_stream, 0);
}

extern "C" int fitrig_detect_batch(fitrig_ctx* c, float tau, fitrig_candidate* h_out, int64_t capacity, int64_t* n_found,
                                   int64_t* n_found_per_stack, void* cuda_stream) {
  if (!n_found_per_stack) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_batch: n_found_per_stack is NULL");
  return detect_core(c, tau, h_out, capacity, n_found, n_found_per_stack, cuda_stream, 0);
}

extern "C" int fitrig_detect_launch(fitrig_ctx* c, float tau, int64_t capacity, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_launch: ctx is NULL");
  if (capacity < 0) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_launch: capacity < 0");
  return detect_launch_core(c, tau, capacity, cuda_stream, 0);
}

extern "C" int fitrig_detect_fetch(fitrig_ctx* c, fitrig_candidate* h_out, int64_t* n_found, int64_t* n_found_per_stack) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_fetch: ctx is NULL");
  if (!n_found) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_fetch: n_found is NULL");
  return detect_fetch_core(c, h_out, n_found, n_found_per_stack);
}

// Eq. 10 for the current map: magnitude spectra, eta, k*, and the statistics of eta
static int launch_spectrum(fitrig_ctx* c, cudaStream_t st, double* shard_out) {
  const bool chained = !c->tune.no_pdl;
  SpectrumParams sp;
  sp.q = c->q; sp.tw = c->tw; sp.eta = c->eta; sp.kstar = c->kstar; sp.nt = (int)c->nt; sp.U = c->U; sp.B = c->B;
  sp.mag = c->mag; sp.harmonics = c->prm.harmonics;
  sp.nblk = c->spec_nblk; sp.chunk = kSpecChunk; sp.parts = c->sparts; sp.counters = c->scounter; sp.mu = c->smu; sp.sigma = c->ssigma;
  sp.shard_out = shard_out;
  if (c->U / 2 >= 1) {
    const dim3 grid((unsigned)((c->nt * c->B + 127) / 128), (unsigned)((c->U / 2 + kDftBins - 1) / kDftBins));
    CUDA_TRY(launch_chain(dft_mag_kernel, grid, dim3(128), sizeof(double2) * c->U, st, chained, sp));
    c->launches++;
  }
  const int grid = (int)std::min<long long>((long long)c->spec_nblk * c->B, 8ll * c->num_sms);
  CUDA_TRY(launch_chain(spectrum_kernel, dim3(grid), dim3(kSpecChunk), 0, st, chained, sp));
  c->launches++;
  c->eta_valid = true;
  return FITRIG_OK;
}

static int detect_launch_core(fitrig_ctx* c, float tau, int64_t capacity, void* cuda_stream, int unit_offset) {
  if (!(tau == tau)) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect: sigma_threshold is NaN");
  if (!c->have_map) return fail(FITRIG_ERR_STATE, "fitrig_detect: no current map (call fitrig_tlisi or fitrig_stream first)");
  if (c->detect_launched - c->detect_fetched >= 2)
    return fail(FITRIG_ERR_STATE, "fitrig_detect_launch: two detections are in flight; fetch one first");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  const bool freq = c->prm.branch == FITRIG_BRANCH_FREQUENCY;
  if (freq && !c->eta_valid) {
    int rc = launch_spectrum(c, st, nullptr);
    if (rc) return rc;
  }
  DetectSlot& d = c->slot[c->detect_launched & 1];
  const long long rows = freq ? c->B : (long long)c->B * c->U;
  const long long N = rows * c->nt;
  const long long want = std::min<long long>(capacity, N);
  if (want > d.cand_cap) {  // grow the device list (rare: only for very low thresholds)
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaFree(d.cand_dev));
    d.cand_dev = nullptr;
    d.cand_cap = 0;
    CUDA_TRY(cudaMalloc(&d.cand_dev, sizeof(fitrig_candidate) * want));
    d.cand_cap = want;
  }
  CompactParams cp;
  cp.v = freq ? c->eta : c->q;
  cp.raw = c->raw; cp.kstar = c->kstar;
  cp.mu = freq ? c->smu : c->mu; cp.sigma = freq ? c->ssigma : c->sigma;
  cp.tau = tau; cp.rows = (int)rows; cp.rows_per_batch = freq ? 1 : c->U; cp.nt = c->nt;
  cp.Tx = c->Tx; cp.Ty = c->Ty; cp.H = c->H; cp.W = c->W; cp.tile = c->prm.tile; cp.stride = c->prm.stride; cp.branch = c->prm.branch;
  cp.row_offset = c->prm.row_offset;
  cp.unit_offset = unit_offset;
  cp.pix8 = c->map_pix8;
  cp.out = reinterpret_cast<fitrig_candidate*>(d.cand_dev);
  cp.cap = std::min<long long>(d.cand_cap, std::max<long long>(capacity, 0));
  cp.host_total = reinterpret_cast<unsigned long long*>(d.cand_host_dev);
  cp.host_out = reinterpret_cast<fitrig_candidate*>(d.cand_host_dev + sizeof(CandHeader));
  cp.host_cap = std::min<long long>(cp.cap, kHostStageCands);
  cp.host_offsets = d.counts_host_dev; cp.B = c->B;
  cp.status = c->cstatus; cp.ticket = c->cticket; cp.ticket_base = c->ticket_base;
  if (++c->compact_epoch == 0) c->compact_epoch = 1;
  cp.epoch = c->compact_epoch;
  const int threads = 512;
  const long long per_min = 4 * threads;  // a block is worth launching for at least this many entries
  int grid = (int)std::min<long long>(c->compact_grid_max, (N + per_min - 1) / per_min);
  grid = std::max(grid, 1);
  cp.seg = ((N + grid - 1) / grid + threads - 1) / threads * threads;
  CUDA_TRY(launch_chain(compact_kernel, dim3(grid), dim3(threads), 0, st, !c->tune.no_pdl, cp));
  c->ticket_base += (unsigned)grid;
  c->launches++;
  CUDA_TRY(cudaEventRecord(d.done, st));
  d.stream = st; d.pending = true; d.cap = cp.cap; d.host_cap = cp.host_cap;
  c->detect_launched++;
  return FITRIG_OK;
}

static int detect_fetch_core(fitrig_ctx* c, fitrig_candidate* h_out, int64_t* n_found, int64_t* n_per_stack) {
  if (c->detect_launched == c->detect_fetched) return fail(FITRIG_ERR_STATE, "fitrig_detect_fetch: nothing was launched");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  DetectSlot& d = c->slot[c->detect_fetched & 1];
  // the kernel has written the count and the first kHostStageCands candidates straight into mapped pinned memory
  // (no copy in the stream); a copy from the device list only for longer lists
  CUDA_TRY(cudaEventSynchronize(d.done));
  const long long total = (long long)reinterpret_cast<CandHeader*>(d.cand_host)->total;
  const long long nwrite = std::min<long long>(total, d.cap);
  if (nwrite > 0 && !h_out)  // (the launch stays unfetched: a call with a proper buffer still gets its result)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_detect_fetch: h_out is NULL and there are %lld candidates to deliver", nwrite);
  c->detect_fetched++;  // from here on the result counts as delivered and the slot is free for the next launch
  d.pending = false;
  const long long n1 = std::min(nwrite, d.host_cap);
  if (n1 > 0) memcpy(h_out, d.cand_host + sizeof(CandHeader), sizeof(fitrig_candidate) * n1);
  if (nwrite > n1) {  // (a later launch writes the other slot's list: this one is still intact)
    CUDA_TRY(cudaMemcpy(h_out + n1, reinterpret_cast<fitrig_candidate*>(d.cand_dev) + n1,
                        sizeof(fitrig_candidate) * (nwrite - n1), cudaMemcpyDeviceToHost));
  }
  *n_found = total;
  if (n_per_stack)  // the kernel reports how many candidates precede each stack; the counts are the differences
    for (int b = 0; b < c->B; ++b) {
      const long long lo = b == 0 ? 0 : (long long)d.counts_host[b];
      const long long hi = b + 1 < c->B ? (long long)d.counts_host[b + 1] : total;
      n_per_stack[b] = hi - lo;
    }
  if (total > d.cap)
    return fail(FITRIG_ERR_CAPACITY, "fitrig_detect: %lld candidates, capacity %lld", total, (long long)d.cap);
  return FITRIG_OK;
}

// ---------------------------------------------------------------------------------------------
// sub-tile localisation (R28)
// ---------------------------------------------------------------------------------------------
template <typename T>
struct DevBuf {  // a device allocation that frees itself on every return path
  T* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  cudaError_t alloc(size_t n) { return cudaMalloc(&p, sizeof(T) * std::max<size_t>(n, 1)); }
};

extern "C" int fitrig_localise(fitrig_ctx* c, const fitrig_candidate* h_cands, int64_t n, int32_t method, int32_t oversample,
                               const float* h_eta, fitrig_position* h_out, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: ctx is NULL");
  if (n < 0 || (n > 0 && (!h_cands || !h_out))) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: NULL argument");
  if (method < 0 || method > 3) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: unknown method %d", method);
  if (oversample < 1 || oversample > 8) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: oversample must be 1 .. 8");
  if (c->prm.branch != FITRIG_BRANCH_FREQUENCY || c->B != 1)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: needs a frequency-branch context without batch");
  if (!h_eta && !c->eta_valid) return fail(FITRIG_ERR_STATE, "fitrig_localise: no eta yet (call fitrig_detect first)");
  if (n == 0) return FITRIG_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  const int tile = c->prm.tile;
  std::vector<int2> tiles(n);
  for (int64_t k = 0; k < n; ++k) {
    const int x = h_cands[k].x, y = h_cands[k].y - c->prm.row_offset;
    if (x < 0 || x >= c->W || y < 0 || y >= c->H) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_localise: candidate %lld is outside the image", (long long)k);
    tiles[k] = make_int2(x / tile, y / tile);
  }
  // eta as doubles
  std::vector<float> ef(c->nt);
  if (h_eta) memcpy(ef.data(), h_eta, sizeof(float) * c->nt);
  else {
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaMemcpy(ef.data(), c->eta, sizeof(float) * c->nt, cudaMemcpyDeviceToHost));
  }
  std::vector<double> ed(ef.begin(), ef.end());
  const int side = 2 * tile * oversample + 1;
  const size_t per_cand = (size_t)3 * side * c->Ty;  // doubles of scratch per candidate
  const int64_t chunk = std::max<int64_t>(1, std::min<int64_t>(n, (int64_t)((256ull << 20) / (per_cand * 8))));
  DevBuf<double> d_eta, d_rowm, d_scr;
  DevBuf<int2> d_tiles;
  DevBuf<fitrig_position> d_out;
  CUDA_TRY(d_eta.alloc(c->nt));
  CUDA_TRY(d_rowm.alloc(c->nt));
  CUDA_TRY(d_scr.alloc(std::max<size_t>((size_t)c->nt, per_cand * chunk)));
  CUDA_TRY(d_tiles.alloc(chunk));
  CUDA_TRY(d_out.alloc(chunk));
  CUDA_TRY(cudaMemcpyAsync(d_eta.p, ed.data(), sizeof(double) * c->nt, cudaMemcpyHostToDevice, st));
  LocaliseParams lp;
  lp.eta = d_eta.p; lp.rowm = d_rowm.p; lp.scratch = d_scr.p; lp.tiles = d_tiles.p; lp.out = d_out.p;
  lp.Ty = c->Ty; lp.Tx = c->Tx; lp.tile = tile; lp.method = method; lp.oversample = oversample; lp.n = 0;
  if (method == FITRIG_INTERP_SPLINE) {
    spline_rows_kernel<<<(c->Ty + 63) / 64, 64, 0, st>>>(lp);
    CUDA_TRY(cudaGetLastError());
    c->launches++;
  }
  for (int64_t k0 = 0; k0 < n; k0 += chunk) {
    const int m = (int)std::min<int64_t>(chunk, n - k0);
    lp.n = m;
    CUDA_TRY(cudaMemcpyAsync(d_tiles.p, tiles.data() + k0, sizeof(int2) * m, cudaMemcpyHostToDevice, st));
    localise_kernel<<<m, 128, 0, st>>>(lp);
    CUDA_TRY(cudaGetLastError());
    c->launches++;
    CUDA_TRY(cudaMemcpyAsync(h_out + k0, d_out.p, sizeof(fitrig_position) * m, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
  }
  if (c->prm.row_offset)
    for (int64_t k = 0; k < n; ++k) h_out[k].y += (double)c->prm.row_offset;
  return FITRIG_OK;
}

// ---------------------------------------------------------------------------------------------
// real-time mode (timeline of Fig. 14)
// ---------------------------------------------------------------------------------------------
extern "C" int fitrig_push_reset(fitrig_ctx* c) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push_reset: ctx is NULL");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  if (c->push_key) CUDA_TRY(cudaMemset(c->push_key, 0, sizeof(unsigned)));
  if (c->push_ring) {  // an empty cube
    CUDA_TRY(cudaMemset(c->raw, 0, sizeof(RawTile) * c->nmap));
    if (c->raw_blocks) CUDA_TRY(cudaMemset(c->raw_blocks, 0, sizeof(RawTile) * (size_t)c->B * c->U * c->Cy * c->Cx));
  }
  c->push_count = 0;
  c->push_next = 0;
  for (int i = 0; i < kPushSlots; ++i) c->push_free_pending[i] = false;
  return FITRIG_OK;
}

extern "C" int fitrig_push(fitrig_ctx* c, const float* snapshot, float tau, float* d_tlisi, fitrig_candidate* h_out,
                           int64_t capacity, int64_t* n_found, int64_t* unit, void* cuda_stream) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push: ctx is NULL");
  if (!n_found || !unit) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push: n_found or unit is NULL");
  const bool freq = c->prm.branch == FITRIG_BRANCH_FREQUENCY;
  if (c->prm.accumulate != 1 || c->B != 1 || c->prm.stride != c->prm.tile)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push: no accumulation, no batch, no overlapping windows");
  if (!freq && c->L != 3)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push: image branch: create the context with n_snapshots = 3 (one unit per push)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  const long long img = (long long)c->H * c->W;
  if (!c->push_ring) {
    CUDA_TRY(cudaMalloc(&c->push_ring, sizeof(float) * img * kPushSlots));
    CUDA_TRY(cudaMalloc(&c->push_key, sizeof(unsigned)));
    CUDA_TRY(cudaMemset(c->push_key, 0, sizeof(unsigned)));
    CUDA_TRY(cudaMemset(c->raw, 0, sizeof(RawTile) * c->nmap));
    if (c->raw_blocks) CUDA_TRY(cudaMemset(c->raw_blocks, 0, sizeof(RawTile) * (size_t)c->B * c->U * c->Cy * c->Cx));
    for (int i = 0; i < kPushSlots; ++i) {
      CUDA_TRY(cudaEventCreateWithFlags(&c->ev_push_copied[i], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&c->ev_push_free[i], cudaEventDisableTiming));
    }
    if (!c->copy_stream) CUDA_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    if (!c->ev_entry) CUDA_TRY(cudaEventCreateWithFlags(&c->ev_entry, cudaEventDisableTiming));
  }
  *unit = -1;
  *n_found = 0;
  // (1) the new snapshot starts its way to the device (host pinned memory, or a device pointer) ...
  if (snapshot) {
    const int slot = (int)(c->push_count % kPushSlots);
    CUDA_TRY(cudaEventRecord(c->ev_entry, st));  // the copy may not overtake work already queued by the caller
    CUDA_TRY(cudaStreamWaitEvent(c->copy_stream, c->ev_entry, 0));
    if (c->push_free_pending[slot]) CUDA_TRY(cudaStreamWaitEvent(c->copy_stream, c->ev_push_free[slot], 0));
    CUDA_TRY(cudaMemcpyAsync(c->push_ring + (long long)slot * img, snapshot, sizeof(float) * img, cudaMemcpyDefault,
                             c->copy_stream));
    c->copies++;
    CUDA_TRY(cudaEventRecord(c->ev_push_copied[slot], c->copy_stream));
  }
  // (2) ... while the unit whose three snapshots were pushed BEFORE this call is computed (Fig. 14: copy of
  // snapshot n+3 overlaps trigger kernel n)
  const long long n = c->push_next;
  int rc = FITRIG_OK;
  if (n + 3 <= c->push_count) {
    for (int k = 0; k < 3; ++k) CUDA_TRY(cudaStreamWaitEvent(st, c->ev_push_copied[(n + k) % kPushSlots], 0));
    RowsOpt opt;
    opt.z0 = (int)(n % kPushSlots); opt.zmod = kPushSlots; opt.key = c->push_key;
    opt.units = 1;
    opt.row0 = (int)(n % c->U);  // image branch: U = 1; frequency branch: the cube is a ring of the last U tile matrices
    rc = launch_tlisi_rows(c, c->push_ring, img, c->H, 0, true, st, opt);
    if (rc) return rc;
    CUDA_TRY(cudaEventRecord(c->ev_push_free[n % kPushSlots], st));  // x_n is not needed again
    c->push_free_pending[n % kPushSlots] = true;
    // M = running maximum over x_0 .. x_{n+2} (R24): every matrix of the cube is (re)normalised by it
    c->fin_user_row = freq ? opt.row0 : -1;  // d_tlisi receives the newest tile matrix
    rc = launch_finalize(c, d_tlisi, st, c->push_key);
    c->fin_user_row = -1;
    if (rc) return rc;
    if (n + 1 > 0x7fffffffll) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_push: unit index overflow");
    if (!freq || n + 1 >= c->U) {  // frequency branch: Eq. 10-12 once the cube holds U units (R29)
      rc = detect_core(c, tau, h_out, capacity, n_found, nullptr, cuda_stream, freq ? 0 : (int)n);
      if (rc != FITRIG_OK && rc != FITRIG_ERR_CAPACITY) return rc;
    } else {
      CUDA_TRY(cudaStreamSynchronize(st));
    }
    *unit = n;
    c->push_next = n + 1;
  }
  if (snapshot) c->push_count++;
  return rc;
}

// ---------------------------------------------------------------------------------------------
// row shards
// ---------------------------------------------------------------------------------------------
static int shard_check(fitrig_ctx* c, const char* who) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "%s: ctx is NULL", who);
  if (c->B != 1) return fail(FITRIG_ERR_INVALID_ARG, "%s: not with params.batch > 1", who);
  if (!c->have_map) return fail(FITRIG_ERR_STATE, "%s: no current map (call fitrig_tlisi first)", who);
  return FITRIG_OK;
}

extern "C" int fitrig_shard_export(fitrig_ctx* c, double* d_out, void* cuda_stream) {
  int rc = shard_check(c, "fitrig_shard_export");
  if (rc) return rc;
  if (!d_out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_shard_export: d_out is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  ShardExportParams ep;
  ep.raw = c->raw; ep.gmax_key = c->gmax_key + c->key_idx; ep.out = d_out;
  ep.H = c->H; ep.W = c->W; ep.tile = c->prm.tile; ep.stride = c->prm.stride; ep.Ty = c->Ty; ep.Tx = c->Tx; ep.U = c->U;
  ep.nblk = c->fin_nblk; ep.chunk = c->fin_chunk; ep.parts = c->parts; ep.counters = c->counters;
  ep.pix8 = c->map_pix8;
  CUDA_TRY(launch_chain(shard_export_kernel, dim3(c->fin_grid), dim3(256), 0, st, !c->tune.no_pdl, ep));
  c->launches++;
  return FITRIG_OK;
}

extern "C" int fitrig_shard_import(fitrig_ctx* c, const double* d_all, int32_t world, float* d_tlisi, void* cuda_stream) {
  int rc = shard_check(c, "fitrig_shard_import");
  if (rc) return rc;
  if (!d_all || world < 1) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_shard_import: d_all is NULL or world < 1");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  FinalizeParams fp;
  fill_finalize_params(c, &fp, d_tlisi, c->gmax_key + c->key_idx);
  fp.gmax_key_next = nullptr;  // (the finalise of fitrig_tlisi has prepared the next call's key already)
  fp.shard_all = d_all; fp.shard_world = world;
  CUDA_TRY(launch_chain(c->map_pix8 ? finalize_kernel<true> : finalize_kernel<false>, dim3(c->fin_grid), dim3(256), 0, st, false, fp));
  c->launches++;
  c->eta_valid = false;
  return FITRIG_OK;
}

extern "C" int fitrig_shard_export_eta(fitrig_ctx* c, double* d_out, void* cuda_stream) {
  int rc = shard_check(c, "fitrig_shard_export_eta");
  if (rc) return rc;
  if (!d_out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_shard_export_eta: d_out is NULL");
  if (c->prm.branch != FITRIG_BRANCH_FREQUENCY)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_shard_export_eta: the context is not in the frequency branch");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  return launch_spectrum(c, (cudaStream_t)cuda_stream, d_out);
}

extern "C" int fitrig_shard_import_eta(fitrig_ctx* c, const double* d_all, int32_t world, void* cuda_stream) {
  int rc = shard_check(c, "fitrig_shard_import_eta");
  if (rc) return rc;
  if (!d_all || world < 1) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_shard_import_eta: d_all is NULL or world < 1");
  if (c->prm.branch != FITRIG_BRANCH_FREQUENCY || !c->eta_valid)
    return fail(FITRIG_ERR_STATE, "fitrig_shard_import_eta: call fitrig_shard_export_eta first (frequency branch)");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  shard_import_eta_kernel<<<1, 32, 0, (cudaStream_t)cuda_stream>>>(d_all, world, c->smu, c->ssigma);
  CUDA_TRY(cudaGetLastError());
  c->launches++;
  return FITRIG_OK;
}

// ---------------------------------------------------------------------------------------------
// getters
// ---------------------------------------------------------------------------------------------
extern "C" int fitrig_get_stats(const fitrig_ctx* c, float* M, double* mu, double* sigma) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_get_stats: ctx is NULL");
  if (!c->have_map) return fail(FITRIG_ERR_STATE, "fitrig_get_stats: no current map");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  if (M) CUDA_TRY(cudaMemcpy(M, c->M_dev, sizeof(float) * c->B, cudaMemcpyDeviceToHost));
  const bool freq_stats = c->prm.branch == FITRIG_BRANCH_FREQUENCY && c->eta_valid;
  const size_t R = (size_t)c->B * c->U;
  if (mu) CUDA_TRY(cudaMemcpy(mu, c->mu, sizeof(double) * R, cudaMemcpyDeviceToHost));
  if (sigma) CUDA_TRY(cudaMemcpy(sigma, c->sigma, sizeof(double) * R, cudaMemcpyDeviceToHost));
  if (freq_stats) {  // eta's statistics take the place of unit 0's in every stack
    std::vector<double> m(c->B), sd(c->B);
    CUDA_TRY(cudaMemcpy(m.data(), c->smu, sizeof(double) * c->B, cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(sd.data(), c->ssigma, sizeof(double) * c->B, cudaMemcpyDeviceToHost));
    for (int b = 0; b < c->B; ++b) {
      if (mu) mu[(size_t)b * c->U] = m[b];
      if (sigma) sigma[(size_t)b * c->U] = sd[b];
    }
  }
  return FITRIG_OK;
}

extern "C" int fitrig_get_map(const fitrig_ctx* c, int32_t which, float* h_out) {
  if (!c || !h_out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_get_map: NULL argument");
  if (!c->have_map) return fail(FITRIG_ERR_STATE, "fitrig_get_map: no current map");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  switch (which) {
    case 0: CUDA_TRY(cudaMemcpy(h_out, c->q, sizeof(float) * c->nmap, cudaMemcpyDeviceToHost)); break;
    case 1: CUDA_TRY(cudaMemcpy(h_out, c->tlisi, sizeof(float) * c->nmap, cudaMemcpyDeviceToHost)); break;
    case 2:
    case 3: {
      if (c->prm.branch != FITRIG_BRANCH_FREQUENCY || !c->eta_valid)
        return fail(FITRIG_ERR_STATE, "fitrig_get_map: eta needs the frequency branch and a previous fitrig_detect");
      const long long ne = c->nt * c->B;
      if (which == 2) {
        CUDA_TRY(cudaMemcpy(h_out, c->eta, sizeof(float) * ne, cudaMemcpyDeviceToHost));
      } else {
        std::vector<int> k(ne);
        CUDA_TRY(cudaMemcpy(k.data(), c->kstar, sizeof(int) * ne, cudaMemcpyDeviceToHost));
        for (long long i = 0; i < ne; ++i) h_out[i] = (float)k[i];
      }
      break;
    }
    default: return fail(FITRIG_ERR_INVALID_ARG, "fitrig_get_map: which = %d", which);
  }
  return FITRIG_OK;
}

extern "C" int fitrig_get_raw(const fitrig_ctx* c, float* sumD, float* maxD, float* sumR, int32_t* ax, int32_t* ay) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_get_raw: ctx is NULL");
  if (!c->have_map) return fail(FITRIG_ERR_STATE, "fitrig_get_raw: no current map");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  std::vector<RawTile> r(c->nmap);
  if (c->map_pix8) {  // tiles of one pixel: 8-byte records {Delta, r}
    std::vector<RawPix> px(c->nmap);
    CUDA_TRY(cudaMemcpy(px.data(), c->raw, sizeof(RawPix) * c->nmap, cudaMemcpyDeviceToHost));
    for (long long i = 0; i < c->nmap; ++i) { r[i].sumD = px[i].delta; r[i].maxD = px[i].delta; r[i].sumR = px[i].r; r[i].pos = 0; }
  } else {
    CUDA_TRY(cudaMemcpy(r.data(), c->raw, sizeof(RawTile) * c->nmap, cudaMemcpyDeviceToHost));
  }
  const int tile = c->prm.tile, stride = c->prm.stride;
  for (long long i = 0; i < c->nmap; ++i) {
    const long long t = i % c->nt;
    const int ty = (int)(t / c->Tx), tx = (int)(t % c->Tx);
    if (sumD) sumD[i] = r[i].sumD;
    if (maxD) maxD[i] = r[i].maxD;
    if (sumR) sumR[i] = r[i].sumR;
    if (ax) ax[i] = tx * stride + r[i].pos % tile;
    if (ay) ay[i] = ty * stride + r[i].pos / tile;
  }
  return FITRIG_OK;
}

extern "C" int fitrig_profile(fitrig_ctx* c, int32_t enable) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_profile: ctx is NULL");
  c->profile = enable != 0;
  c->ev_used = 0;
  c->fin_used = 0;
  return FITRIG_OK;
}

extern "C" int fitrig_last_timing(const fitrig_ctx* c, float* main_ms, int32_t* main_launches, float* fin_ms,
                                  int32_t* fin_launches) {
  if (!c) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_last_timing: ctx is NULL");
  if (!c->profile || !c->have_map) return fail(FITRIG_ERR_STATE, "fitrig_last_timing: profiling was not enabled");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  float tot = 0.f;
  for (int i = 0; i < c->ev_used; ++i) {
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]));
    tot += ms;
  }
  if (main_ms) *main_ms = tot;
  if (main_launches) *main_launches = c->ev_used;
  float ftot = 0.f;
  for (int i = 0; i < c->fin_used; ++i) {
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, c->fin_pool[2 * i], c->fin_pool[2 * i + 1]));
    ftot += ms;
  }
  if (fin_ms) *fin_ms = ftot;
  if (fin_launches) *fin_launches = c->fin_used;
  fitrig_ctx* m = const_cast<fitrig_ctx*>(c);  // reading starts a new accumulation window
  m->ev_used = 0;
  m->fin_used = 0;
  return FITRIG_OK;
}

extern "C" int fitrig_probe_read_bandwidth(fitrig_ctx* c, const void* d_buf, int64_t bytes, int32_t reps, float* gbs,
                                           void* cuda_stream) {
  if (!c || !d_buf || !gbs) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_probe_read_bandwidth: NULL argument");
  if (bytes < 16 || reps < 1 || ((uintptr_t)d_buf % 16) != 0)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_probe_read_bandwidth: need a 16-byte aligned buffer of at least 16 bytes, reps >= 1");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(c->prm.device));
  struct EventPair {  // destroyed on every return path
    cudaEvent_t a = nullptr, b = nullptr;
    ~EventPair() {
      if (a) cudaEventDestroy(a);
      if (b) cudaEventDestroy(b);
    }
  } ev;
  CUDA_TRY(cudaEventCreate(&ev.a));
  CUDA_TRY(cudaEventCreate(&ev.b));
  const cudaEvent_t e0 = ev.a, e1 = ev.b;
  float best = 0.f;
  const long long n4 = bytes / 16;
  for (int r = 0; r < reps + 1; ++r) {  // the first pass warms up
    CUDA_TRY(cudaEventRecord(e0, st));
    read_probe_kernel<<<c->num_sms * 4, 512, 0, st>>>(reinterpret_cast<const float4*>(d_buf), n4, c->M_dev);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(e1, st));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    if (r > 0 && ms > 0.f) best = std::max(best, (float)((double)n4 * 16.0 / (ms * 1e-3) / 1e9));
  }
  *gbs = best;
  return FITRIG_OK;
}

extern "C" int fitrig_choose_accumulate(const float* d_stack, int32_t H, int32_t W, int32_t L, float eps, int32_t g_max, int32_t device,
                                        int32_t* g_out, double* contrast, int32_t* n_levels, void* cuda_stream) {
  if (!d_stack || !g_out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate: NULL argument");
  if (H < 1 || W < 1 || L < 3 || g_max < 1 || device < 0 || !(eps == eps))
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate: need H, W >= 1, n_snapshots >= 3 (PAPER.md:155), g_max >= 1, a threshold");
  int ndev = 0;
  CUDA_TRY(cudaGetDeviceCount(&ndev));
  if (device >= ndev) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate: device %d of %d", device, ndev);
  CUDA_TRY(cudaSetDevice(device));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, device));
  if (prop.major < 10) return fail(FITRIG_ERR_CUDA, "fitrig_choose_accumulate: this library is built for sm_100a (B200) only");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int levels = 0;
  for (int g = 1; levels < kAccumLevels && g <= g_max && L / g >= 3; g *= 2) ++levels;  // admissible group sizes (R30)
  const long long hw = (long long)H * W;
  const int nblocks = (int)std::min<long long>((hw + 255) / 256, 8ll * prop.multiProcessorCount);
  DevBuf<double2> parts;
  DevBuf<AccumChoice> choice;
  CUDA_TRY(parts.alloc((size_t)levels * nblocks));
  CUDA_TRY(choice.alloc(1));
  for (int lv = 0; lv < levels; ++lv) {
    accum_contrast_kernel<<<nblocks, 256, 0, st>>>(d_stack, hw, L, 1 << lv, parts.p + (size_t)lv * nblocks);
    CUDA_TRY(cudaGetLastError());
  }
  accum_choose_kernel<<<1, 256, 0, st>>>(parts.p, nblocks, levels, L, hw, eps, choice.p);
  CUDA_TRY(cudaGetLastError());
  AccumChoice h;
  CUDA_TRY(cudaMemcpyAsync(&h, choice.p, sizeof(h), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  *g_out = h.g;
  if (n_levels) *n_levels = h.n_levels;
  if (contrast)
    for (int i = 0; i < h.n_levels; ++i) contrast[i] = h.contrast[i];
  return FITRIG_OK;
}

// ---------------------------------------------------------------------------------------------
// fitrig_choose_accumulate_static -- the same rule for callers that must not allocate (see fitrig.h).  The block
// partials and the decision record live in ONE file-scope device array instead of two cudaMalloc'ed buffers; the same
// two kernels run on it with the same grid, so the contrasts come out bit-identical to fitrig_choose_accumulate's.
//
// g_static_accum below is, in host code, only a handle for the runtime: its host-side address is NOT where the GPU
// keeps the array.  The launches therefore get the device address that cudaGetSymbolAddress returns, looked up once
// per device (with that device current) and cached.  Every CUDA device that loads this library carries its own copy of
// the array (sizeof(StaticAccumScratch), about 128 KB) until the process exits.
// ---------------------------------------------------------------------------------------------
static_assert(FITRIG_STATIC_ACCUM_MAX_PARTIALS >= kAccumLevels * 8 * 148, "one B200 with all six levels must fit");

struct StaticAccumScratch {
  AccumChoice choice;  // decision record, cleared at the start of every call
  unsigned char pad[256 - sizeof(AccumChoice)];
  double2 partials[FITRIG_STATIC_ACCUM_MAX_PARTIALS];  // [level][block]; every entry a call reads, that call wrote first
};
static __device__ __align__(256) StaticAccumScratch g_static_accum;

static const int kStaticAccumMaxDevices = 64;
struct StaticAccumDevice {
  StaticAccumScratch* scratch;  // DEVICE address of g_static_accum on this device; NULL until the set-up has run
  int num_sms;
};
static StaticAccumDevice g_static_accum_dev[kStaticAccumMaxDevices];
static std::mutex g_static_accum_mu;

// Once per device, with `device` current: which GPU this is and where its copy of the array lives.
static int static_accum_setup(int device, StaticAccumDevice* out) {
  std::lock_guard<std::mutex> lock(g_static_accum_mu);
  StaticAccumDevice& d = g_static_accum_dev[device];
  if (!d.scratch) {
    int major = 0, sms = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    if (major < 10) return fail(FITRIG_ERR_CUDA, "fitrig_choose_accumulate_static: this library is built for sm_100a (B200) only");
    void* addr = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&addr, g_static_accum));
    if (!addr) return fail(FITRIG_ERR_CUDA, "fitrig_choose_accumulate_static: cudaGetSymbolAddress returned no address on device %d", device);
    d.num_sms = sms;
    d.scratch = static_cast<StaticAccumScratch*>(addr);
  }
  *out = d;
  return FITRIG_OK;
}

extern "C" int fitrig_choose_accumulate_static(const float* d_stack, int32_t H, int32_t W, int32_t L, float eps, int32_t g_max,
                                               int32_t device, int32_t* g_out, double* contrast, int32_t* n_levels,
                                               void* cuda_stream) {
  if (!d_stack || !g_out) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate_static: NULL argument");
  if (H < 1 || W < 1 || L < 3 || g_max < 1 || device < 0 || !(eps == eps))
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate_static: need H, W >= 1, n_snapshots >= 3 (PAPER.md:155), g_max >= 1, a threshold");
  int ndev = 0;
  CUDA_TRY(cudaGetDeviceCount(&ndev));
  if (device >= ndev || device >= kStaticAccumMaxDevices)
    return fail(FITRIG_ERR_INVALID_ARG, "fitrig_choose_accumulate_static: device %d of %d (at most %d)", device, ndev, kStaticAccumMaxDevices);
  CUDA_TRY(cudaSetDevice(device));
  StaticAccumDevice dev;
  if (int rc = static_accum_setup(device, &dev)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int levels = 0;
  for (int g = 1; levels < kAccumLevels && g <= g_max && L / g >= 3; g *= 2) ++levels;  // admissible group sizes (R30)
  const long long hw = (long long)H * W;
  const int nblocks = (int)std::min<long long>((hw + 255) / 256, 8ll * dev.num_sms);  // as fitrig_choose_accumulate
  if ((long long)levels * nblocks > FITRIG_STATIC_ACCUM_MAX_PARTIALS)
    return fail(FITRIG_ERR_INVALID_ARG,
                "fitrig_choose_accumulate_static: %d levels x %d blocks = %lld partial sums, the static scratch holds %d "
                "(lower g_max, or use fitrig_choose_accumulate, which allocates what it needs)",
                levels, nblocks, (long long)levels * nblocks, FITRIG_STATIC_ACCUM_MAX_PARTIALS);
  // The array still holds what the previous call left.  The partials need no clearing (each level's kernel writes all
  // `nblocks` entries that the decision kernel then reads); the decision record is cleared so that nothing of an
  // earlier call can be read back as this call's answer.
  CUDA_TRY(cudaMemsetAsync(&dev.scratch->choice, 0, 256, st));
  for (int lv = 0; lv < levels; ++lv) {
    accum_contrast_kernel<<<nblocks, 256, 0, st>>>(d_stack, hw, L, 1 << lv, dev.scratch->partials + (size_t)lv * nblocks);
    CUDA_TRY(cudaGetLastError());
  }
  accum_choose_kernel<<<1, 256, 0, st>>>(dev.scratch->partials, nblocks, levels, L, hw, eps, &dev.scratch->choice);
  CUDA_TRY(cudaGetLastError());
  AccumChoice h;
  CUDA_TRY(cudaMemcpyAsync(&h, &dev.scratch->choice, sizeof(h), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (h.n_levels < 1 || h.n_levels > levels)
    return fail(FITRIG_ERR_CUDA, "fitrig_choose_accumulate_static: no decision came back (did another call use the scratch at the same time?)");
  *g_out = h.g;
  if (n_levels) *n_levels = h.n_levels;
  if (contrast)
    for (int i = 0; i < h.n_levels; ++i) contrast[i] = h.contrast[i];
  return FITRIG_OK;
}

extern "C" int fitrig_stream_timeline(const fitrig_ctx* c, float* ms, int32_t capacity, int32_t* n_strips) {
  if (!c || !n_strips) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream_timeline: NULL argument");
  if (capacity < 0 || (capacity > 0 && !ms)) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_stream_timeline: bad ms/capacity");
  *n_strips = c->tl_strips;
  if (c->tl_strips == 0) return fail(FITRIG_ERR_STATE, "fitrig_stream_timeline: no fitrig_stream ran under fitrig_profile(1)");
  CUDA_TRY(cudaSetDevice(c->prm.device));
  CUDA_TRY(cudaDeviceSynchronize());
  for (int i = 0; i < std::min(capacity, c->tl_strips); ++i)
    for (int k = 0; k < 4; ++k)
      CUDA_TRY(cudaEventElapsedTime(&ms[4 * i + k], c->tl_pool[0], c->tl_pool[4 * i + k]));
  return FITRIG_OK;
}

extern "C" int fitrig_launch_count(const fitrig_ctx* c, int64_t* n) {
  if (!c || !n) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_launch_count: NULL argument");
  *n = c->launches;
  return FITRIG_OK;
}

extern "C" int fitrig_copy_count(const fitrig_ctx* c, int64_t* n) {
  if (!c || !n) return fail(FITRIG_ERR_INVALID_ARG, "fitrig_copy_count: NULL argument");
  *n = c->copies;
  return FITRIG_OK;
}
