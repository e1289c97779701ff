// qs_noalloc.cu — qs_matvec_noalloc: y = M x on free rings (C2) through the K1 pair sweep WITHOUT any allocation.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  The sweep's scratch memory - padded copies of r, z, x, the bounding boxes of the blocks of 32 rings, the FP64
// accumulators the sweep reduces into and its work counter, which every other entry point carves out of a workspace
// that qs_init allocates - lives in ONE file-scope `static __device__` array of fixed size (kScratchBytes, 544 KB for
// at most QS_NOALLOC_MAX_RINGS = 16,384 rings); every GPU that loads the library holds it until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address.  The device address is taken once per
// device, with that device current, by cudaGetSymbolAddress (setup_device below, return code checked) and it is that
// pointer the kernels receive.
//
// Every call shares the array, which keeps the previous call's contents: the set-up kernel rewrites all inputs and
// clears the accumulators and the work counter at the start of each call.  Calls that OVERLAP on the GPU (two streams,
// two host threads) race on it: the caller serialises them.  The entry point enqueues three kernels on the caller's
// stream and returns; it calls no cudaMalloc, cudaFree, or allocating library routine, and does not synchronise.
#include <mutex>

#include "../../include/qs.h"
#include "qs_internal.h"

namespace qs {
namespace {

constexpr int kMaxRings = QS_NOALLOC_MAX_RINGS;            // multiple of 32
constexpr int kMaxBlocks = kMaxRings / 32;
// layout in doubles: r, z, x, yacc [kMaxRings each] | bbox [kMaxBlocks x 4] | work counter [32 = 256 bytes]
constexpr size_t kOffR = 0, kOffZ = kMaxRings, kOffX = 2 * kMaxRings, kOffY = 3 * kMaxRings;
constexpr size_t kOffBox = 4 * kMaxRings, kOffCounter = kOffBox + 4 * kMaxBlocks;
constexpr size_t kScratchDoubles = kOffCounter + 32;
constexpr size_t kScratchBytes = kScratchDoubles * sizeof(double);   // 557,312 bytes

static __device__ __align__(256) double g_noalloc_scratch[kScratchDoubles];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double* g_scratch_ptr[kMaxDevices] = {};   // device address of g_noalloc_scratch on each device (nullptr: not set up)
int g_sm_count_dev[kMaxDevices] = {};

// once per device, with that device current: the DEVICE address of the static array
int setup_device(int dev, double** ptr, int* sm_count) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (g_scratch_ptr[dev] == nullptr) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_noalloc_scratch);
    if (e != cudaSuccess || p == nullptr)
      return set_error(QS_ERR_CUDA, "qs_matvec_noalloc: cudaGetSymbolAddress of the static scratch array failed");
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
    g_sm_count_dev[dev] = sms;
    g_scratch_ptr[dev] = p;
  }
  *ptr = g_scratch_ptr[dev];
  *sm_count = g_sm_count_dev[dev];
  return QS_OK;
}

__device__ __forceinline__ double wmax(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double wmin(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// One CTA.  Rewrites everything a call reads from the scratch array: padded r, z, x (padding: far-away dummy rings that
// carry no current, as qs_init pads), the block boxes, zeroed accumulators and work counter.
constexpr int kPrepThreads = 1024;
__global__ void __launch_bounds__(kPrepThreads) noalloc_prepare_kernel(int n, int np, const double* __restrict__ r,
                                                                       const double* __restrict__ z,
                                                                       const double* __restrict__ x,
                                                                       double* __restrict__ scratch) {
  __shared__ double part[kPrepThreads / 32];
  __shared__ double zmax_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double zm = -1e300;
  for (int i = threadIdx.x; i < n; i += kPrepThreads) zm = fmax(zm, z[i]);
  zm = wmax(zm);
  if (lane == 0) part[warp] = zm;
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = part[0];
    for (int k = 1; k < kPrepThreads / 32; ++k) m = fmax(m, part[k]);
    zmax_s = m;
  }
  __syncthreads();
  const double zmax = zmax_s, r0 = r[0];
  double* sr = scratch + kOffR;
  double* sz = scratch + kOffZ;
  double* sx = scratch + kOffX;
  double* sy = scratch + kOffY;
  double4* box = reinterpret_cast<double4*>(scratch + kOffBox);
  for (int b = warp; b < np / 32; b += kPrepThreads / 32) {   // one warp per block of 32 rings
    const int i = 32 * b + lane;
    const bool in = i < n;
    const double ri = in ? r[i] : r0;
    const double zi = in ? z[i] : zmax + 1.0 + 0.01 * (i - n);
    sr[i] = ri;
    sz[i] = zi;
    sx[i] = in ? x[i] : 0.0;
    sy[i] = 0.0;
    const double rlo = wmin(ri), rhi = wmax(ri), zlo = wmin(zi), zhi = wmax(zi);
    if (lane == 0) box[b] = make_double4(rlo, rhi, zlo, zhi);
  }
  if (threadIdx.x < 32) scratch[kOffCounter + threadIdx.x] = 0.0;   // the 64-bit work counter (all-zero bits)
}

__global__ void noalloc_finish_kernel(int n, const double* __restrict__ yacc, double scale, double* __restrict__ y) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) y[i] = scale * yacc[i];
}

}  // namespace
}  // namespace qs

extern "C" int qs_matvec_noalloc(int32_t n_rings, const double* d_r, const double* d_z, double softening,
                                 const double* d_x, double* d_y, void* stream) {
  using namespace qs;
  if (n_rings < 0) return set_error(QS_ERR_ARG, "qs_matvec_noalloc: n_rings < 0");
  if (n_rings > kMaxRings)
    return set_error(QS_ERR_ARG, "qs_matvec_noalloc: n_rings exceeds QS_NOALLOC_MAX_RINGS (16384): the static scratch "
                                 "array is fixed-size; use qs_init + qs_matvec_device for larger ring sets");
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return set_error(QS_ERR_CUDA, "qs_matvec_noalloc: no CUDA device (libqs has no CPU path)");
  if (dev < 0 || dev >= kMaxDevices) return set_error(QS_ERR_ARG, "qs_matvec_noalloc: device ordinal out of range");
  double* scratch = nullptr;
  int sm_count = 148;
  const int rc = setup_device(dev, &scratch, &sm_count);
  if (rc != QS_OK) return rc;
  if (n_rings == 0) return QS_OK;   // set-up only
  if (!d_r || !d_z || !d_x || !d_y) return set_error(QS_ERR_ARG, "qs_matvec_noalloc: NULL array");
  if (!(softening > 0.0)) return set_error(QS_ERR_ARG, "qs_matvec_noalloc: softening must be > 0");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int np = (n_rings + 31) / 32 * 32, nb = np / 32;
  noalloc_prepare_kernel<<<1, kPrepThreads, 0, st>>>(n_rings, np, d_r, d_z, d_x, scratch);
  SweepParams prm;
  prm.r = scratch + kOffR;
  prm.z = scratch + kOffZ;
  prm.x = scratch + kOffX;
  prm.cur = scratch + kOffX;
  prm.bbox = reinterpret_cast<const double4*>(scratch + kOffBox);
  prm.yacc = scratch + kOffY;
  prm.bracc = nullptr;
  prm.bzacc = nullptr;
  prm.counter = reinterpret_cast<unsigned long long*>(scratch + kOffCounter);
  prm.done = nullptr;
  prm.nb = nb;
  prm.n_items = sweep_items(nb, false);
  prm.soft_all = softening * softening;   // free rings: dz^2 + g^2 for ALL pairs (C2)
  prm.soft_self = 0.0;
  prm.minsep2 = 0.0;
  prm.diag_d2 = prm.soft_all;
  const int wpc = sweep_warps_per_cta();
  int grid = sweep_grid(sm_count, false, nb);
  const long long need = (prm.n_items + wpc - 1) / wpc;
  if (need < grid) grid = static_cast<int>(need);
  const long long warps = static_cast<long long>(grid) * wpc;
  const long long per = prm.n_items / (warps * 8);
  prm.chunk = static_cast<int>(per < 1 ? 1 : (per > 32 ? 32 : per));
  cudaError_t e = launch_sweep(prm, false, grid, st);
  if (e == cudaSuccess) {
    const int fgrid = (n_rings + 255) / 256;
    noalloc_finish_kernel<<<fgrid, 256, 0, st>>>(n_rings, scratch + kOffY, 0.5 * kMu0 * kPi, d_y);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return set_error(QS_ERR_CUDA, cudaGetErrorString(e));
  return QS_OK;
}
