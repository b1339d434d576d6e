// csrc/gamer_hydro_api.cu — the C ABI declared in include/gamer_hydro.h: argument validation, TMA descriptor
// encoding, kernel selection and launch. No torch types, no CPU fallback: without a compute-capability-10
// device every compute entry point returns an error.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <mutex>

#include "../../include/gamer_hydro.h"
#include "hydro_fused.cuh"
#include "hydro_generic.cuh"
#include "hydro_f2.cuh"
#include "hydro_duo.cuh"
#include "hydro_zpair.cuh"
#include "hydro_aux.cuh"
#include "hydro_rtvd.cuh"

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct State {
  bool ready = false;
  int device = -1;
  int sm_count = 0;
  int smem_per_sm = 0;
  unsigned long long* status = nullptr;  // [0] guard cells, [1] non-positive outputs, [2 ..] per-call reduction slots
  void* scratch = nullptr;               // generic path: FS + FL for `scratch_groups` groups
  size_t scratch_bytes = 0;
  cudaEvent_t scratch_free = nullptr;    // recorded after the last reader of the scratch: the next user waits on it
  bool scratch_used = false;
  // host-buffer path
  cudaStream_t hstream[3] = {nullptr, nullptr, nullptr};
  void* hbuf_in[3] = {nullptr, nullptr, nullptr};
  void* hbuf_out[3] = {nullptr, nullptr, nullptr};
  void* hbuf_bf[3] = {nullptr, nullptr, nullptr};
  size_t hbuf_groups = 0;
  int hbuf_N = 0, hbuf_ghost = 0;
  void* grid_buf = nullptr;              // gamer_hydro_advance: second ghosted array for the fused-halo ping-pong
  size_t grid_buf_bytes = 0;
  int path = GAMER_HYDRO_PATH_AUTO;
  char cuda_msg[256] = "no CUDA error recorded";
  EncodeTiledFn encode = nullptr;
};

State g_state;
std::mutex g_mutex;
std::atomic<unsigned long long> g_launches{0};

constexpr int kReduceSlots = 64;    // signal-speed maxima of concurrent max_speed / advance calls
unsigned long long g_slot_busy = 0; // bit s set: slot s is leased (under g_mutex)

// Every call that reduces a signal-speed maximum on the device and READS it back leases its own 8-byte slot for as
// long as it runs (gamer_hydro_advance: for all its steps), so calls on other threads and streams can neither zero
// it nor add their maxima to it. With all 64 leased the call fails with GAMER_HYDRO_BUSY instead of sharing a slot.
// Slot kReduceSlots is a sink nobody reads (the public gamer_hydro_step_grid, which returns before its kernel ran).
struct SlotLease {
  int idx = -1;
  SlotLease() {
    std::lock_guard<std::mutex> lk(g_mutex);
    for (int s = 0; s < kReduceSlots; ++s)
      if (!(g_slot_busy >> s & 1ull)) { g_slot_busy |= 1ull << s; idx = s; break; }
  }
  ~SlotLease() {
    if (idx < 0) return;
    std::lock_guard<std::mutex> lk(g_mutex);
    g_slot_busy &= ~(1ull << idx);
  }
  SlotLease(const SlotLease&) = delete;
  SlotLease& operator=(const SlotLease&) = delete;
  bool ok() const { return idx >= 0; }
  unsigned long long* ptr() const { return g_state.status + 2 + idx; }
};
unsigned long long* sink_reduce_slot() { return g_state.status + 2 + kReduceSlots; }

constexpr int kGenericChunk = 512;  // groups per generic-path launch (bounds the scratch buffer)

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_state.cuda_msg, sizeof(g_state.cuda_msg), "%s: %s", what, cudaGetErrorString(e));
  return GAMER_HYDRO_CUDA_ERROR;
}
#define CK(call)                                        \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

template <class R, int LIM, bool Fast>
int set_fused_attr() {
  CK(cudaFuncSetAttribute(gh::fused_kernel<R, LIM, Fast, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                          gh::FusedSmem<R>::total));
  CK(cudaFuncSetAttribute(gh::fused_kernel<R, LIM, Fast, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                          gh::FusedSmem<R>::total));
  return 0;
}

int init_locked(int device) {
  if (g_state.ready && g_state.device == device) return 0;
  if (g_state.ready) return GAMER_HYDRO_INVALID_ARG;  // one device per process
  int count = 0;
  CK(cudaGetDeviceCount(&count));
  if (device < 0 || device >= count) return GAMER_HYDRO_INVALID_ARG;
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) return GAMER_HYDRO_NOT_SM100;
  CK(cudaSetDevice(device));
  g_state.sm_count = prop.multiProcessorCount;
  g_state.smem_per_sm = (int)prop.sharedMemPerMultiprocessor;
  // [0] guard cells, [1] non-positive outputs, [2 ..] leased reduction slots, then one sink slot
  CK(cudaMalloc(&g_state.status, (2 + kReduceSlots + 1) * sizeof(unsigned long long)));
  CK(cudaMemset(g_state.status, 0, (2 + kReduceSlots + 1) * sizeof(unsigned long long)));
  CK(cudaEventCreateWithFlags(&g_state.scratch_free, cudaEventDisableTiming));
  int rc;
  if ((rc = set_fused_attr<float, 0, true>())) return rc;
  if ((rc = set_fused_attr<float, 1, true>())) return rc;
  if ((rc = set_fused_attr<float, 2, true>())) return rc;
  if ((rc = set_fused_attr<double, 0, false>())) return rc;
  if ((rc = set_fused_attr<double, 1, false>())) return rc;
  if ((rc = set_fused_attr<double, 2, false>())) return rc;
  CK(cudaFuncSetAttribute(gh::zpair_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::ZSmem::total));
  CK(cudaFuncSetAttribute(gh::zpair_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::ZSmem::total));
  CK(cudaFuncSetAttribute(gh::zpair_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::ZSmem::total));
  CK(cudaFuncSetAttribute(gh::duo_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::duo_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::duo_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::duo_halo_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::duo_halo_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::duo_halo_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::DHALVES * gh::DuoSmem::total_padded));
  CK(cudaFuncSetAttribute(gh::rtvd_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::RtvdSmem::total));
  CK(cudaFuncSetAttribute(gh::rtvd_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, gh::RtvdSmem::total));
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
  if (qres != cudaDriverEntryPointSuccess || fn == nullptr) {
    snprintf(g_state.cuda_msg, sizeof(g_state.cuda_msg), "cuTensorMapEncodeTiled not available from the driver");
    return GAMER_HYDRO_CUDA_ERROR;
  }
  g_state.encode = reinterpret_cast<EncodeTiledFn>(fn);
  g_state.device = device;
  g_state.ready = true;
  return 0;
}

int ensure_init() {
  std::lock_guard<std::mutex> lk(g_mutex);
  if (g_state.ready) return 0;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  return init_locked(dev);
}

// grows the generic-path scratch; g_mutex must be HELD (a grow frees the old buffer: nobody may read the pointer or
// enqueue work on it meanwhile)
int ensure_scratch_locked(size_t bytes) {
  if (g_state.scratch_bytes >= bytes) return 0;
  if (g_state.scratch) {
    CK(cudaDeviceSynchronize());
    CK(cudaFree(g_state.scratch));
    g_state.scratch = nullptr;
    g_state.scratch_bytes = 0;
  }
  CK(cudaMalloc(&g_state.scratch, bytes));
  g_state.scratch_bytes = bytes;
  return 0;
}

int ensure_scratch(size_t bytes) {
  std::lock_guard<std::mutex> lk(g_mutex);
  return ensure_scratch_locked(bytes);
}

template <class R>
size_t generic_scratch_bytes(int groups, int N, int ghost) {
  const gh::GenericShape sh = gh::make_shape(N, ghost);
  return (size_t)groups * (size_t)(sh.fs_stride + sh.fl_stride) * sizeof(R);
}

template <class R>
int validate(const R* U_in, R* U_out, R* bflux, int n_groups, int N, int ghost, R dt, R dx, R gamma, int limiter) {
  if (n_groups < 0 || N < 1 || ghost < 2) return GAMER_HYDRO_INVALID_ARG;
  if (!(dt > R(0)) || !(dx > R(0)) || !isfinite((double)dt) || !isfinite((double)dx)) return GAMER_HYDRO_INVALID_ARG;
  if (!(gamma > R(1)) || !isfinite((double)gamma)) return GAMER_HYDRO_INVALID_ARG;
  if (limiter != GAMER_HYDRO_MINMOD && limiter != GAMER_HYDRO_VANLEER && limiter != GAMER_HYDRO_MC)
    return GAMER_HYDRO_INVALID_ARG;
  if (n_groups == 0) return 0;
  if (!U_in || !U_out) return GAMER_HYDRO_INVALID_ARG;
  if (((uintptr_t)U_in & 15) || ((uintptr_t)U_out & 15) || ((uintptr_t)bflux & 15)) return GAMER_HYDRO_INVALID_ARG;
  return 0;
}

template <class R>
bool fused_supported(int N, int ghost) {
  // TMA: every global stride and the byte offset of the box start along x must be multiples of 16 bytes
  // (measured on B200: a box starting at x = 1 float raises "illegal instruction").
  const int S = N + 2 * ghost;
  return N == gh::FN && ((S * (int)sizeof(R)) % 16 == 0) && (((ghost - 2) * (int)sizeof(R)) % 16 == 0);
}

// rank-5 tensor map (x, y, z, var, group) over U_in; box = box_z consecutive z planes of all five variables
// (20 x 20 x box_z x 5 x 1); planes outside the array are zero-filled
template <class R>
int encode_plane_map(const R* U_in, int n_groups, int N, int ghost, CUtensorMap& map, int box_z = 1) {
  const int S = N + 2 * ghost;
  const cuuint64_t dims[5] = {(cuuint64_t)S, (cuuint64_t)S, (cuuint64_t)S, 5, (cuuint64_t)n_groups};
  const cuuint64_t strides[4] = {(cuuint64_t)S * sizeof(R), (cuuint64_t)S * S * sizeof(R),
                                 (cuuint64_t)S * S * S * sizeof(R), (cuuint64_t)5 * S * S * S * sizeof(R)};
  const cuuint32_t box[5] = {(cuuint32_t)gh::FS, (cuuint32_t)gh::FS, (cuuint32_t)box_z, 5, 1};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  const CUtensorMapDataType dt_ = sizeof(R) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  CUresult r = g_state.encode(&map, dt_, 5, const_cast<R*>(U_in), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_state.cuda_msg, sizeof(g_state.cuda_msg), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return GAMER_HYDRO_CUDA_ERROR;
  }
  return 0;
}

template <class R, int LIM, bool VAR>
void launch_fused_one(int grid, int smem, cudaStream_t stream, const CUtensorMap& map, R* U_out, R* bflux, int n_groups,
                      int goff, const gh::GasConst<R>& c, int flags, R* midflux) {
  constexpr bool Fast = sizeof(R) == 4;
  gh::fused_kernel<R, LIM, Fast, VAR><<<grid, gh::FNT, smem, stream>>>(map, U_out, bflux, n_groups, goff, c,
                                                                         g_state.status, flags, midflux);
}

template <class R>
int launch_fused(const R* U_in, R* U_out, R* bflux, int n_groups, int N, int ghost, R dt, R dx, R gamma, int limiter,
                 cudaStream_t stream, int flags = 0, R* midflux = nullptr) {
  CUtensorMap map;
  int rc = encode_plane_map<R>(U_in, n_groups, N, ghost, map);
  if (rc) return rc;
  const gh::GasConst<R> c = gh::make_consts<R>(dt, dx, gamma);
  const int smem = gh::FusedSmem<R>::total;
  // persistent CTAs: as many as are resident at once (shared memory decides: 2 per SM in fp32, 1 in fp64)
  const int per_sm = (2 * smem + 2048 <= g_state.smem_per_sm && gh::FMINB >= 2) ? 2 : 1;
  const int resident = g_state.sm_count * per_sm;
  const int grid = n_groups < resident ? n_groups : resident;
  const bool var = flags != 0 || midflux != nullptr;
#define GH_FUSED(LIM)                                                                                               \
  (var ? launch_fused_one<R, LIM, true>(grid, smem, stream, map, U_out, bflux, n_groups, ghost - 2, c, flags, midflux) \
       : launch_fused_one<R, LIM, false>(grid, smem, stream, map, U_out, bflux, n_groups, ghost - 2, c, 0, nullptr))
  if (limiter == 0) GH_FUSED(0);
  else if (limiter == 1) GH_FUSED(1);
  else GH_FUSED(2);
#undef GH_FUSED
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

// fp32 performance path: one cell per thread, the f32x2 lanes carry two directions of the cell (hydro_duo.cuh)
int launch_duo(const float* U_in, float* U_out, float* bflux, int n_groups, int N, int ghost, float dt, float dx,
               float gamma, int limiter, cudaStream_t stream, const gh::HaloGrid* halo = nullptr) {
  CUtensorMap map;
  int rc = encode_plane_map<float>(U_in, n_groups, N, ghost, map);
  if (rc) return rc;
  const gh::PairConst c = gh::make_pair_consts(dt, dx, gamma);
  const int smem = gh::DHALVES * gh::DuoSmem::total_padded;   // one CTA per SM: two independent 320-thread halves
  const int want = (n_groups + gh::DHALVES - 1) / gh::DHALVES;
  const int grid = want < g_state.sm_count ? want : g_state.sm_count;
  const int threads = gh::FNT * gh::DHALVES;
  if (halo) {
    if (limiter == 0)
      gh::duo_halo_kernel<0><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status, *halo);
    else if (limiter == 1)
      gh::duo_halo_kernel<1><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status, *halo);
    else
      gh::duo_halo_kernel<2><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status, *halo);
  } else if (limiter == 0) {
    gh::duo_kernel<0><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  } else if (limiter == 1) {
    gh::duo_kernel<1><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  } else {
    gh::duo_kernel<2><<<grid, threads, smem, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  }
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

// fp32 default: one column per thread, the f32x2 lanes carry two consecutive z planes (hydro_zpair.cuh)
int launch_zpair(const float* U_in, float* U_out, float* bflux, int n_groups, int N, int ghost, float dt, float dx,
                 float gamma, int limiter, cudaStream_t stream) {
  CUtensorMap map;
  int rc = encode_plane_map<float>(U_in, n_groups, N, ghost, map, 2);
  if (rc) return rc;
  const gh::PairConst c = gh::make_pair_consts(dt, dx, gamma);
  const int grid = n_groups < g_state.sm_count ? n_groups : g_state.sm_count;   // persistent: one CTA per SM
  if (limiter == 0)
    gh::zpair_kernel<0><<<grid, gh::ZNT, gh::ZSmem::total, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  else if (limiter == 1)
    gh::zpair_kernel<1><<<grid, gh::ZNT, gh::ZSmem::total, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  else
    gh::zpair_kernel<2><<<grid, gh::ZNT, gh::ZSmem::total, stream>>>(map, U_out, bflux, n_groups, ghost - 2, c, g_state.status);
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

template <class R>
int launch_generic(const R* U_in, R* U_out, R* bflux, int n_groups, int N, int ghost, R dt, R dx, R gamma,
                   int limiter, cudaStream_t stream, int flags = 0, R* midflux = nullptr) {
  const int chunk = n_groups < kGenericChunk ? n_groups : kGenericChunk;
  const gh::GenericShape sh = gh::make_shape(N, ghost);
  const gh::GasConst<R> c = gh::make_consts<R>(dt, dx, gamma);
  const long long ne = (long long)sh.E * sh.E * sh.E, nf = 3LL * (N + 1) * N * N, nc = (long long)N * N * N;
  // ONE scratch buffer serves every stream: calls on different streams are chained by an event (the predictor of the
  // next call waits for the update kernel of the previous one). Growing the buffer, reading its address, the wait, the
  // launches and the record all happen under ONE hold of the lock: the chain is a total order, and no other host thread
  // can free and re-allocate the buffer (a larger generic shape) between this call's pointer read and its launches.
  std::lock_guard<std::mutex> lk(g_mutex);
  int rc = ensure_scratch_locked(generic_scratch_bytes<R>(chunk, N, ghost));
  if (rc) return rc;
  R* FS = reinterpret_cast<R*>(g_state.scratch);
  R* FL = FS + (size_t)chunk * sh.fs_stride;
  if (g_state.scratch_used) CK(cudaStreamWaitEvent(stream, g_state.scratch_free, 0));
  for (int g0 = 0; g0 < n_groups; g0 += chunk) {
    const int ng = (n_groups - g0) < chunk ? (n_groups - g0) : chunk;
    const R* in = U_in + (size_t)g0 * sh.in_stride;
    R* out = U_out + (size_t)g0 * sh.out_stride;
    R* bf = bflux ? bflux + (size_t)g0 * 30 * N * N : nullptr;
    const dim3 gp((unsigned)((ne + 127) / 128), ng), gf((unsigned)((nf + 127) / 128), ng),
        gu((unsigned)((nc + 127) / 128), ng);
    R* mf = midflux ? midflux + (size_t)g0 * 15 * N * N : nullptr;
    if (limiter == 0) gh::predict_kernel<R, 0><<<gp, 128, 0, stream>>>(in, FS, sh, c, g_state.status, (long long)g0);
    else if (limiter == 1) gh::predict_kernel<R, 1><<<gp, 128, 0, stream>>>(in, FS, sh, c, g_state.status, (long long)g0);
    else gh::predict_kernel<R, 2><<<gp, 128, 0, stream>>>(in, FS, sh, c, g_state.status, (long long)g0);
    gh::flux_kernel<R><<<gf, 128, 0, stream>>>(FS, FL, bf, sh, c, flags, mf, (long long)g0);
    gh::update_kernel<R><<<gu, 128, 0, stream>>>(in, FL, out, sh, c, g_state.status);
    g_launches.fetch_add(3);
  }
  CK(cudaGetLastError());
  CK(cudaEventRecord(g_state.scratch_free, stream));
  g_state.scratch_used = true;
  return 0;
}

template <class R>
int step_impl(const R* U_in, R* U_out, R* bflux, int n_groups, int N, int ghost, R dt, R dx, R gamma, int limiter,
              cudaStream_t stream, int flags = 0, R* midflux = nullptr) {
  int rc = validate<R>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter);
  if (rc) return rc;
  if (flags < 0 || flags > 3 || ((uintptr_t)midflux & 15) || (midflux && (N & 1))) return GAMER_HYDRO_INVALID_ARG;
  if (n_groups == 0) return 0;
  if ((rc = ensure_init())) return rc;
  int path = g_state.path;
  if (flags != 0 || midflux) {
    // the robustness variants live in the scalar fused kernel (N = 16) and the generic kernels
    if (path != GAMER_HYDRO_PATH_GENERIC && fused_supported<R>(N, ghost))
      return launch_fused<R>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream, flags, midflux);
    return launch_generic<R>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream, flags, midflux);
  }
  if (path == GAMER_HYDRO_PATH_AUTO)
    path = fused_supported<R>(N, ghost) ? GAMER_HYDRO_PATH_FUSED : GAMER_HYDRO_PATH_GENERIC;
  if (path == GAMER_HYDRO_PATH_FUSED || path == GAMER_HYDRO_PATH_FUSED_SCALAR || path == GAMER_HYDRO_PATH_FUSED_DUO) {
    if (!fused_supported<R>(N, ghost)) return GAMER_HYDRO_UNSUPPORTED;
    if constexpr (sizeof(R) == 4) {
      if (path == GAMER_HYDRO_PATH_FUSED)
        return launch_zpair(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
      if (path == GAMER_HYDRO_PATH_FUSED_DUO)
        return launch_duo(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
    }
    return launch_fused<R>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
  }
  return launch_generic<R>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
}

void free_host_bufs() {
  for (int s = 0; s < 3; ++s) {
    if (g_state.hbuf_in[s]) cudaFree(g_state.hbuf_in[s]);
    if (g_state.hbuf_out[s]) cudaFree(g_state.hbuf_out[s]);
    if (g_state.hbuf_bf[s]) cudaFree(g_state.hbuf_bf[s]);
    g_state.hbuf_in[s] = g_state.hbuf_out[s] = g_state.hbuf_bf[s] = nullptr;
  }
  g_state.hbuf_groups = 0;
}

}  // namespace

namespace {

template <class R, class Bits>
int max_speed_impl(const R* U, int n_groups, int N, int ghost, double gamma, double* h_max, cudaStream_t stream) {
  if (!U || !h_max || n_groups < 0 || N < 1 || ghost < 0 || !(gamma > 1.0)) return GAMER_HYDRO_INVALID_ARG;
  *h_max = 0.0;
  if (n_groups == 0) return 0;
  int rc = ensure_init();
  if (rc) return rc;
  SlotLease lease;   // held until the value has been read back (the stream is synchronised below)
  if (!lease.ok()) return GAMER_HYDRO_BUSY;
  Bits* slot = reinterpret_cast<Bits*>(lease.ptr());
  CK(cudaMemsetAsync(slot, 0, sizeof(unsigned long long), stream));
  const long long n_cells = (long long)n_groups * N * N * N;
  const int threads = 256;
  long long want = (n_cells + threads - 1) / threads;
  const int grid = (int)(want < (long long)g_state.sm_count * 16 ? want : (long long)g_state.sm_count * 16);
  if (N == 16 && ghost == 2)
    gh::max_speed_kernel<R, Bits, 16, 2><<<grid, threads, 0, stream>>>(U, n_cells, N, ghost, (R)gamma, slot);
  else
    gh::max_speed_kernel<R, Bits, 0, 0><<<grid, threads, 0, stream>>>(U, n_cells, N, ghost, (R)gamma, slot);
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  Bits bits = 0;
  CK(cudaMemcpyAsync(&bits, slot, sizeof(Bits), cudaMemcpyDeviceToHost, stream));
  CK(cudaStreamSynchronize(stream));
  R v;
  memcpy(&v, &bits, sizeof(R));
  *h_max = (double)v;
  return 0;
}

// want_max: also accumulate the signal-speed maximum of the refilled state into the status slot (zeroed first)
template <class R, class Bits>
int fill_ghosts_impl(const R* U_out, R* U_in, int gx, int gy, int gz, int N, int ghost, int bcx, int bcy, int bcz,
                     cudaStream_t stream, unsigned long long* max_slot = nullptr, double gamma = 5.0 / 3.0) {
  if (!U_out || !U_in || gx < 1 || gy < 1 || gz < 1 || N < 1 || ghost < 0 || (bcx | bcy | bcz) < 0 || bcx > 1 ||
      bcy > 1 || bcz > 1)
    return GAMER_HYDRO_INVALID_ARG;
  if ((long long)gx * gy * gz > 0x7fffffffLL) return GAMER_HYDRO_INVALID_ARG;
  if (ghost > gx * N || ghost > gy * N || ghost > gz * N) return GAMER_HYDRO_UNSUPPORTED;  // shell wider than the box
  int rc = ensure_init();
  if (rc) return rc;
  Bits* slot = nullptr;
  if (max_slot) {
    slot = reinterpret_cast<Bits*>(max_slot);
    CK(cudaMemsetAsync(slot, 0, sizeof(unsigned long long), stream));
  }
  const int grid = gx * gy * gz;   // one CTA per group
  if (N == 16 && ghost == 2)
    // 1024 threads per group: 1.35 ms against 1.63 ms with 256 on the headline grid (5.9 TB/s of the 6.45 measured peak)
    gh::fill_ghosts_kernel<R, Bits, 2, 16, 2><<<grid, 1024, 0, stream>>>(U_out, U_in, gx, gy, gz, N, ghost, bcx, bcy, bcz,
                                                                        (R)gamma, slot);
  else if (N % 2 == 0 && ghost % 2 == 0)
    gh::fill_ghosts_kernel<R, Bits, 2, 0, 0><<<grid, 256, 0, stream>>>(U_out, U_in, gx, gy, gz, N, ghost, bcx, bcy, bcz,
                                                                       (R)gamma, slot);
  else
    gh::fill_ghosts_kernel<R, Bits, 1, 0, 0><<<grid, 256, 0, stream>>>(U_out, U_in, gx, gy, gz, N, ghost, bcx, bcy, bcz,
                                                                       (R)gamma, slot);
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

}  // namespace

extern "C" {

int gamer_hydro_alloc(int max_groups, int N, int ghost, int bytes_per_real, int device) {
  if (max_groups < 0 || N < 1 || ghost < 2 || (bytes_per_real != 4 && bytes_per_real != 8))
    return GAMER_HYDRO_INVALID_ARG;
  {
    std::lock_guard<std::mutex> lk(g_mutex);
    int rc = init_locked(device);
    if (rc) return rc;
  }
  const bool fused = bytes_per_real == 4 ? fused_supported<float>(N, ghost) : fused_supported<double>(N, ghost);
  if (!fused && max_groups > 0) {
    const int chunk = max_groups < kGenericChunk ? max_groups : kGenericChunk;
    const size_t bytes = bytes_per_real == 4 ? generic_scratch_bytes<float>(chunk, N, ghost)
                                             : generic_scratch_bytes<double>(chunk, N, ghost);
    return ensure_scratch(bytes);
  }
  return 0;
}

void gamer_hydro_free(void) {
  std::lock_guard<std::mutex> lk(g_mutex);
  if (!g_state.ready) return;
  cudaDeviceSynchronize();
  free_host_bufs();
  for (int s = 0; s < 3; ++s)
    if (g_state.hstream[s]) { cudaStreamDestroy(g_state.hstream[s]); g_state.hstream[s] = nullptr; }
  if (g_state.scratch) cudaFree(g_state.scratch);
  if (g_state.grid_buf) cudaFree(g_state.grid_buf);
  g_state.grid_buf = nullptr;
  g_state.grid_buf_bytes = 0;
  if (g_state.status) cudaFree(g_state.status);
  g_state.scratch = nullptr;
  g_state.scratch_bytes = 0;
  g_state.status = nullptr;
  g_state.ready = false;
  g_state.device = -1;
}

int gamer_hydro_step(const float* U_in, float* U_out, float* bflux, int n_groups, int N, int ghost, float dt, float dx,
                     float gamma, int limiter, cudaStream_t stream) {
  return step_impl<float>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
}

int gamer_hydro_step_f64(const double* U_in, double* U_out, double* bflux, int n_groups, int N, int ghost, double dt,
                         double dx, double gamma, int limiter, cudaStream_t stream) {
  return step_impl<double>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream);
}

int gamer_hydro_step_ex(const float* U_in, float* U_out, float* bflux, float* midflux, int n_groups, int N, int ghost,
                        float dt, float dx, float gamma, int limiter, int flags, cudaStream_t stream) {
  return step_impl<float>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream, flags, midflux);
}

int gamer_hydro_step_ex_f64(const double* U_in, double* U_out, double* bflux, double* midflux, int n_groups, int N,
                            int ghost, double dt, double dx, double gamma, int limiter, int flags, cudaStream_t stream) {
  return step_impl<double>(U_in, U_out, bflux, n_groups, N, ghost, dt, dx, gamma, limiter, stream, flags, midflux);
}

int gamer_hydro_max_speed(const void* U, int bytes_per_real, int n_groups, int N, int ghost, double gamma,
                          double* h_max, cudaStream_t stream) {
  if (bytes_per_real == 4)
    return max_speed_impl<float, unsigned int>((const float*)U, n_groups, N, ghost, gamma, h_max, stream);
  if (bytes_per_real == 8)
    return max_speed_impl<double, unsigned long long>((const double*)U, n_groups, N, ghost, gamma, h_max, stream);
  return GAMER_HYDRO_INVALID_ARG;
}

int gamer_hydro_fill_ghosts(const void* U_out, void* U_in_with_ghosts, int bytes_per_real, int gx, int gy, int gz, int N,
                            int ghost, int bc_x, int bc_y, int bc_z, cudaStream_t stream) {
  if (bytes_per_real == 4)
    return fill_ghosts_impl<float, unsigned int>((const float*)U_out, (float*)U_in_with_ghosts, gx, gy, gz, N, ghost, bc_x, bc_y, bc_z, stream);
  if (bytes_per_real == 8)
    return fill_ghosts_impl<double, unsigned long long>((const double*)U_out, (double*)U_in_with_ghosts, gx, gy, gz, N, ghost, bc_x, bc_y, bc_z, stream);
  return GAMER_HYDRO_INVALID_ARG;
}

static int step_grid_impl(const float* U, float* U_out, float* bflux, float* U_next, int gx, int gy, int gz, int N,
                          int ghost, float dt, float dx, float gamma, int limiter, cudaStream_t stream,
                          unsigned long long* max_slot) {
  if (gx < 1 || gy < 1 || gz < 1 || (long long)gx * gy * gz > 0x7fffffffLL || !U_next || U_next == U)
    return GAMER_HYDRO_INVALID_ARG;
  const int ng = gx * gy * gz;
  int rc = validate<float>(U, U_out, bflux, ng, N, ghost, dt, dx, gamma, limiter);
  if (rc) return rc;
  if (N != gh::FN || ghost != 2) return GAMER_HYDRO_UNSUPPORTED;   // the fused-halo kernel is the N = 16, ghost = 2 one
  if ((rc = ensure_init())) return rc;
  unsigned int* slot = reinterpret_cast<unsigned int*>(max_slot ? max_slot : sink_reduce_slot());
  CK(cudaMemsetAsync(slot, 0, sizeof(unsigned long long), stream));
  const gh::HaloGrid hg = {U_next, slot, gx, gy, gz};
  return launch_duo(U, U_out, bflux, ng, N, ghost, dt, dx, gamma, limiter, stream, &hg);
}

int gamer_hydro_step_grid(const float* U, float* U_out, float* bflux, float* U_next, int gx, int gy, int gz, int N,
                          int ghost, float dt, float dx, float gamma, int limiter, cudaStream_t stream) {
  return step_grid_impl(U, U_out, bflux, U_next, gx, gy, gz, N, ghost, dt, dx, gamma, limiter, stream, nullptr);
}

int gamer_hydro_advance(float* U, float* U_out, float* bflux, int gx, int gy, int gz, int N, int ghost, int bc_x,
                        int bc_y, int bc_z, int n_steps, float cfl, float dx, float gamma, int limiter, float* h_dts,
                        cudaStream_t stream) {
  if (!U || !U_out || gx < 1 || gy < 1 || gz < 1 || n_steps < 0 || !(cfl > 0.0f) || !(dx > 0.0f))
    return GAMER_HYDRO_INVALID_ARG;
  const long long ng = (long long)gx * gy * gz;
  if (ng > 0x7fffffffLL) return GAMER_HYDRO_INVALID_ARG;
  if (n_steps == 0) return 0;
  if (!(gamma > 1.0f) || N < 1 || ghost < 2) return GAMER_HYDRO_INVALID_ARG;
  double vmax = 0.0;
  int rc = gamer_hydro_max_speed(U, 4, (int)ng, N, ghost, (double)gamma, &vmax, stream);   // state on entry
  if (rc) return rc;
  SlotLease lease;   // this call's own reduction slot for all its steps (every step ends with a synchronised read)
  if (!lease.ok()) return GAMER_HYDRO_BUSY;
  unsigned long long* const slot = lease.ptr();
  // Default: step + ghost refill (the refill pass also accumulates the next signal-speed maximum). With the DUO path
  // selected, a fully periodic grid of 16^3 groups uses the fused-halo variant of that kernel instead: the step
  // kernel itself writes the next step's ghosted array and signal-speed maximum (ping-pong between U and a
  // library-owned second array; that array is shared, so this variant is not re-entrant).
  const bool fused_halo = bc_x == 0 && bc_y == 0 && bc_z == 0 && N == gh::FN && ghost == 2 &&
                          g_state.path == GAMER_HYDRO_PATH_FUSED_DUO;
  const size_t grid_bytes = (size_t)ng * 5 * 20 * 20 * 20 * sizeof(float);
  float* cur = U;
  float* nxt = nullptr;
  if (fused_halo) {
    std::lock_guard<std::mutex> lk(g_mutex);
    if (g_state.grid_buf_bytes < grid_bytes) {
      CK(cudaDeviceSynchronize());
      if (g_state.grid_buf) cudaFree(g_state.grid_buf);
      g_state.grid_buf = nullptr;
      g_state.grid_buf_bytes = 0;
      CK(cudaMalloc(&g_state.grid_buf, grid_bytes));
      g_state.grid_buf_bytes = grid_bytes;
    }
    nxt = (float*)g_state.grid_buf;
  }
  // on ANY exit the caller's U holds the state after the steps completed so far (never a stale ping-pong buffer)
  auto finish = [&](int code) -> int {
    if (cur != U) {
      if (cudaMemcpyAsync(U, cur, grid_bytes, cudaMemcpyDeviceToDevice, stream) != cudaSuccess ||
          cudaStreamSynchronize(stream) != cudaSuccess)
        return code ? code : cuda_fail(cudaGetLastError(), "copy of the final state back to U");
    }
    return code;
  };
  for (int s = 0; s < n_steps; ++s) {
    // no finite positive signal speed (a NaN state reduces to NaN: the device maximum propagates it): invalid state
    if (!(vmax > 0.0) || vmax > 3.0e38) return finish(GAMER_HYDRO_INVALID_ARG);
    const float dt = (float)((double)cfl * (double)dx / vmax);            // R15, fp64 on the host, rounded once (R11)
    if (h_dts) h_dts[s] = dt;
    if (fused_halo) {
      if ((rc = step_grid_impl(cur, U_out, bflux, nxt, gx, gy, gz, N, ghost, dt, dx, gamma, limiter, stream, slot)))
        return finish(rc);
      float* tmp = cur; cur = nxt; nxt = tmp;
    } else {
      if ((rc = gamer_hydro_step(U, U_out, bflux, (int)ng, N, ghost, dt, dx, gamma, limiter, stream))) return finish(rc);
      // ghost refill fused with the signal-speed maximum of the new state (next step's dt)
      if ((rc = fill_ghosts_impl<float, unsigned int>(U_out, U, gx, gy, gz, N, ghost, bc_x, bc_y, bc_z, stream, slot,
                                                      (double)gamma)))
        return finish(rc);
    }
    unsigned int bits = 0;
    if (cudaMemcpyAsync(&bits, slot, sizeof(bits), cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
        cudaStreamSynchronize(stream) != cudaSuccess)
      return finish(cuda_fail(cudaGetLastError(), "read of the signal-speed maximum"));
    float v;
    memcpy(&v, &bits, sizeof(v));
    vmax = (double)v;
  }
  return finish(0);
}

int gamer_hydro_step_host(const float* h_in, float* h_out, float* h_bf, int n_groups, int N, int ghost, float dt,
                          float dx, float gamma, int limiter, int chunk_groups) {
  if (n_groups < 0 || N < 1 || ghost < 2) return GAMER_HYDRO_INVALID_ARG;
  if (n_groups == 0) return 0;
  if (!h_in || !h_out) return GAMER_HYDRO_INVALID_ARG;
  int rc = ensure_init();
  if (rc) return rc;
  const size_t S = (size_t)N + 2 * ghost;
  const size_t in_g = 5 * S * S * S, out_g = (size_t)5 * N * N * N, bf_g = (size_t)30 * N * N;
  if (chunk_groups <= 0) chunk_groups = 256;   // 101 ms per headline step against 104 ms with 1024 (shorter pipeline tail)
  if (chunk_groups > n_groups) chunk_groups = n_groups;
  {
    std::lock_guard<std::mutex> lk(g_mutex);
    if (g_state.hbuf_groups < (size_t)chunk_groups || g_state.hbuf_N != N || g_state.hbuf_ghost != ghost) {
      CK(cudaDeviceSynchronize());
      free_host_bufs();
      for (int s = 0; s < 3; ++s) {
        if (!g_state.hstream[s]) CK(cudaStreamCreateWithFlags(&g_state.hstream[s], cudaStreamNonBlocking));
        CK(cudaMalloc(&g_state.hbuf_in[s], chunk_groups * in_g * sizeof(float)));
        CK(cudaMalloc(&g_state.hbuf_out[s], chunk_groups * out_g * sizeof(float)));
        CK(cudaMalloc(&g_state.hbuf_bf[s], chunk_groups * bf_g * sizeof(float)));
      }
      g_state.hbuf_groups = chunk_groups;
      g_state.hbuf_N = N;
      g_state.hbuf_ghost = ghost;
    }
  }
  int n = 0;
  for (int g0 = 0; g0 < n_groups; g0 += chunk_groups, ++n) {
    const int s = n % 3;
    const int ng = (n_groups - g0) < chunk_groups ? (n_groups - g0) : chunk_groups;
    cudaStream_t st = g_state.hstream[s];
    float* d_in = (float*)g_state.hbuf_in[s];
    float* d_out = (float*)g_state.hbuf_out[s];
    float* d_bf = h_bf ? (float*)g_state.hbuf_bf[s] : nullptr;
    CK(cudaMemcpyAsync(d_in, h_in + (size_t)g0 * in_g, ng * in_g * sizeof(float), cudaMemcpyHostToDevice, st));
    rc = step_impl<float>(d_in, d_out, d_bf, ng, N, ghost, dt, dx, gamma, limiter, st);
    if (rc) return rc;
    CK(cudaMemcpyAsync(h_out + (size_t)g0 * out_g, d_out, ng * out_g * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (h_bf)
      CK(cudaMemcpyAsync(h_bf + (size_t)g0 * bf_g, d_bf, ng * bf_g * sizeof(float), cudaMemcpyDeviceToHost, st));
  }
  for (int s = 0; s < 3; ++s) CK(cudaStreamSynchronize(g_state.hstream[s]));
  return 0;
}

int gamer_rtvd_step(const float* U_in, float* U_out, int n_groups, int N, int ghost, float dt, float dx, float gamma,
                    int sweep, cudaStream_t stream) {
  if (n_groups < 0 || N < 1 || ghost < 3 || (sweep != 0 && sweep != 1)) return GAMER_HYDRO_INVALID_ARG;
  if (!(dt > 0.0f) || !(dx > 0.0f) || !isfinite((double)dt) || !isfinite((double)dx)) return GAMER_HYDRO_INVALID_ARG;
  if (!(gamma > 1.0f) || !isfinite((double)gamma)) return GAMER_HYDRO_INVALID_ARG;
  if (n_groups == 0) return 0;
  if (!U_in || !U_out || ((uintptr_t)U_in & 15) || ((uintptr_t)U_out & 15)) return GAMER_HYDRO_INVALID_ARG;
  if (N != gh::RN || ghost != gh::RG) return GAMER_HYDRO_UNSUPPORTED;   // the kernel holds one 22^3 x 5 tile per CTA
  int rc = ensure_init();
  if (rc) return rc;
  const gh::RtvdConst c = {dt / dx, 0.5f * (dt / dx), gamma - 1.0f, gamma};
  const int grid = n_groups < g_state.sm_count ? n_groups : g_state.sm_count;   // persistent: one CTA per SM
  if (sweep == 0) gh::rtvd_kernel<0><<<grid, gh::RNT, gh::RtvdSmem::total, stream>>>(U_in, U_out, n_groups, c);
  else gh::rtvd_kernel<1><<<grid, gh::RNT, gh::RtvdSmem::total, stream>>>(U_in, U_out, n_groups, c);
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

int gamer_hydro_status(unsigned long long* guard_cells, unsigned long long* nonpositive_out) {
  int rc = ensure_init();
  if (rc) return rc;
  unsigned long long h[2];
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(h, g_state.status, sizeof(h), cudaMemcpyDeviceToHost));
  CK(cudaMemset(g_state.status, 0, sizeof(h)));
  if (guard_cells) *guard_cells = h[0];
  if (nonpositive_out) *nonpositive_out = h[1];
  return 0;
}

int gamer_hydro_set_path(int path) {
  if (path < GAMER_HYDRO_PATH_AUTO || path > GAMER_HYDRO_PATH_FUSED_DUO) return GAMER_HYDRO_INVALID_ARG;
  g_state.path = path;
  return 0;
}

int gamer_hydro_set_guard_map(unsigned char* device_map) {
  int rc = ensure_init();
  if (rc) return rc;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpyToSymbol(gh::gh_guard_map, &device_map, sizeof(device_map)));
  return 0;
}

int gamer_hydro_set_hlle_map(unsigned char* device_map) {
  int rc = ensure_init();
  if (rc) return rc;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpyToSymbol(gh::gh_hlle_map, &device_map, sizeof(device_map)));
  return 0;
}

}  // extern "C" (re-opened below, after the no-allocation section)

// ---------------------------------------------------------------------------------------------------------------
// gamer_hydro_max_speed_noalloc: the CFL signal-speed maximum (R15) for callers that must not trigger a device
// allocation. Who that is: an AMR code that sized its patch pools to fill the GPU at start-up (a cudaMalloc issued by
// this library in the middle of a run can then fail for lack of memory, long after the run began), and a time loop
// that keeps copies and kernels of several streams in flight (cudaMalloc and cudaFree wait for the whole device, so an
// allocation inside the loop stalls every one of those streams). gamer_hydro_max_speed goes through the library's
// set-up, which allocates the status block its reduction slot lives in; this variant keeps its partial maxima in the
// fixed array below instead and writes the result to a device address the caller supplies.
//
// The array is part of the loaded library image: every GPU that loads libgamer_hydro.so holds these 256.25 KiB until
// the process exits, whether or not this entry point is ever called. All calls on a device share it and it keeps
// whatever the last call left in it.
constexpr int kNoAllocMaxGroups = 65536;   // twice the headline batch of BASELINE.json:configs[3]
constexpr int kNoAllocHeader = 64;         // words: [0] = number of CTAs that have published their maximum
constexpr int kNoAllocMaxDevices = 64;
static __device__ __align__(256) unsigned int g_noalloc_scratch[kNoAllocHeader + kNoAllocMaxGroups];

namespace {

// One CTA per patch group: maximum of |vx| + |vy| + |vz| + 3 c_s over the group's interior cells (the arithmetic of
// gh::max_speed_kernel, same NaN rule: a NaN cell makes the maximum NaN) -> scratch[header + group]. The CTA that
// publishes last (ticket in scratch[0], which must be 0 when the kernel starts) reduces the per-group maxima and
// writes *d_max. `scratch` is the DEVICE address of g_noalloc_scratch, looked up by the host (see below).
template <int NC, int GC>
__global__ void max_speed_noalloc_kernel(const float* __restrict__ U, int N_rt, int ghost_rt, float gamma,
                                         unsigned int* scratch, float* __restrict__ d_max) {
  const int N = NC > 0 ? NC : N_rt, ghost = NC > 0 ? GC : ghost_rt;
  const int S = N + 2 * ghost;
  const long long S3 = (long long)S * S * S;
  const float* Ug = U + (long long)blockIdx.x * 5 * S3;
  __shared__ float red[32];
  __shared__ bool last;
  auto nanmax = [](float a, float b) { return (b > a || b != b) ? b : a; };
  auto block_max = [&](float m) -> float {   // valid in thread 0
    for (int o = 16; o > 0; o >>= 1) m = nanmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
      m = threadIdx.x < ((blockDim.x + 31) >> 5) ? red[threadIdx.x] : 0.0f;
      for (int o = 16; o > 0; o >>= 1) m = nanmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    }
    __syncthreads();
    return m;
  };
  float m = 0.0f;
  for (int r = threadIdx.x; r < N * N * N; r += blockDim.x) {
    const int i = r % N, j = (r / N) % N, k = r / (N * N);
    const float* p = Ug + ((long long)(k + ghost) * S + (j + ghost)) * S + (i + ghost);
    const float rho = p[0], mx = p[S3], my = p[2 * S3], mz = p[3 * S3], E = p[4 * S3];
    const float ir = 1.0f / rho;
    float P = (gamma - 1.0f) * (E - 0.5f * (mx * mx + my * my + mz * mz) * ir);
    P = P > 0.0f ? P : 0.0f;
    const float v = (fabsf(mx) + fabsf(my) + fabsf(mz)) * ir + 3.0f * sqrtf(gamma * P * ir);
    m = nanmax(m, v);
  }
  m = block_max(m);
  if (threadIdx.x == 0) {
    scratch[kNoAllocHeader + blockIdx.x] = __float_as_uint(m);
    __threadfence();                                        // the maximum is visible before the ticket is
    last = atomicAdd(scratch, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  const volatile unsigned int* part = scratch + kNoAllocHeader;   // written by other CTAs: read past L1
  m = 0.0f;
  for (int g = threadIdx.x; g < (int)gridDim.x; g += blockDim.x) m = nanmax(m, __uint_as_float(part[g]));
  m = block_max(m);
  if (threadIdx.x == 0) *d_max = m;
}

std::mutex g_noalloc_mutex;
unsigned int* g_noalloc_addr[kNoAllocMaxDevices] = {};   // per device: DEVICE address of g_noalloc_scratch, 0 = not set up

// In host code the name g_noalloc_scratch is only a handle for the symbol, not an address the GPU can use, and every
// device that loads the library has its own copy of the array at its own address. Hence: once per device, with that
// device current, ask the runtime where the copy lives, and hand that pointer to the kernel.
int noalloc_scratch_of_current_device(unsigned int** out) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return GAMER_HYDRO_UNSUPPORTED;
  std::lock_guard<std::mutex> lk(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {
    int major = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return GAMER_HYDRO_NOT_SM100;
    void* p = nullptr;
    CK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return GAMER_HYDRO_CUDA_ERROR;
    g_noalloc_addr[dev] = static_cast<unsigned int*>(p);
  }
  *out = g_noalloc_addr[dev];
  return 0;
}

}  // namespace

extern "C" {

int gamer_hydro_max_speed_noalloc_limit(void) { return kNoAllocMaxGroups; }

int gamer_hydro_max_speed_noalloc(const float* U, int n_groups, int N, int ghost, float gamma, float* d_max,
                                  cudaStream_t stream) {
  if (!U || !d_max || n_groups < 1 || N < 1 || ghost < 0 || !(gamma > 1.0f) || ((uintptr_t)d_max & 3))
    return GAMER_HYDRO_INVALID_ARG;
  if (n_groups > kNoAllocMaxGroups) return GAMER_HYDRO_TOO_LARGE;   // the fixed array has one word per group
  unsigned int* scratch = nullptr;
  int rc = noalloc_scratch_of_current_device(&scratch);
  if (rc) return rc;
  // the ticket must start at zero, whatever the previous call (or a call that died half-way) left behind
  CK(cudaMemsetAsync(scratch, 0, sizeof(unsigned int), stream));
  if (N == 16 && ghost == 2)
    max_speed_noalloc_kernel<16, 2><<<n_groups, 256, 0, stream>>>(U, N, ghost, gamma, scratch, d_max);
  else
    max_speed_noalloc_kernel<0, 0><<<n_groups, 256, 0, stream>>>(U, N, ghost, gamma, scratch, d_max);
  g_launches.fetch_add(1);
  CK(cudaGetLastError());
  return 0;
}

unsigned long long gamer_hydro_launch_count(void) { return g_launches.load(); }

const char* gamer_hydro_strerror(int code) {
  switch (code) {
    case GAMER_HYDRO_OK: return "success";
    case GAMER_HYDRO_INVALID_ARG: return "invalid argument";
    case GAMER_HYDRO_UNSUPPORTED: return "unsupported shape for the requested kernel path";
    case GAMER_HYDRO_CUDA_ERROR: return g_state.cuda_msg;
    case GAMER_HYDRO_NOT_SM100: return "device is not compute capability 10.x (sm_100a required)";
    case GAMER_HYDRO_BUSY:
      return "all 64 signal-speed reduction slots are leased by gamer_hydro_max_speed / gamer_hydro_advance calls in flight";
    case GAMER_HYDRO_TOO_LARGE:
      return "batch exceeds the fixed scratch array of gamer_hydro_max_speed_noalloc (65536 patch groups at most): "
             "split the batch or call gamer_hydro_max_speed";
    default: return "unknown error code";
  }
}

}  // extern "C"
