// emm_noalloc.cu -- emm_check_delta_static: the convergence measure of [R9] (L385-387) with NO allocation of any kind.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// It is a variant of the reduction the run driver uses (k_check_reduce + k_check_final, emm_kernels.cu): warp shuffle +
// block reduction, one partial sum per block left in scratch memory, the partials added in a fixed order.  The run driver
// carves that scratch from the caller's workspace; here it is a file-scope device array of a fixed, modest size:
//
//   g_check_part   kStaticMaxSrc x 6 components x 2 sums x kCheckBlocks doubles = 16 * 6 * 2 * 148 * 8 B = 227 328 B
//
// Every GPU that loads the library holds these 222 KB until the process exits.  All calls share the array, and it keeps
// the contents of the last call.  Nothing in it has to start at zero: every slot a call reads has been written by that
// same call (each block writes its own slot, the final kernel reads exactly the slots of the blocks that were launched),
// so no clearing is done.  Calls that overlap on the GPU (different streams, or different host threads on one device) RACE
// on the array; calls on one stream are ordered and safe.
//
// In host code the name `g_check_part` is a host-side stand-in, not a device address: handing it to a kernel faults or,
// where the GPU can reach host memory, silently uses the wrong memory.  The device address is looked up once per device,
// with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels receive.
#include "emm_kernels.cuh"

namespace emm {

namespace {

constexpr int kStaticMaxSrc = EMM_CHECK_STATIC_MAX_NSRC;
constexpr size_t kStaticDoubles = (size_t)kStaticMaxSrc * 6 * 2 * kCheckBlocks;

static __device__ __align__(256) double g_check_part[kStaticDoubles];

// sums of |now - prev|^2 and |now|^2 over the check set, per (source, component): one partial pair per block.
// Unlike k_check_reduce this variant leaves `prev` alone (inputs are const) and knows no run state.
__global__ void __launch_bounds__(256) k_check_reduce_static(const int nchk, const double2 *__restrict__ now, const double2 *__restrict__ prev,
                                                             double *__restrict__ part) {
  const int src = blockIdx.z, c = blockIdx.y;
  double num = 0.0, den = 0.0;
  const size_t base = ((size_t)src * 6 + c) * nchk;
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < nchk; p += gridDim.x * blockDim.x) {
    const double2 a = now[base + p], b = prev[base + p];
    const double dx = a.x - b.x, dy = a.y - b.y;
    num += dx * dx + dy * dy;
    den += a.x * a.x + a.y * a.y;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    num += __shfl_xor_sync(0xffffffffu, num, o);
    den += __shfl_xor_sync(0xffffffffu, den, o);
  }
  __shared__ double sn[32], sd[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { sn[wid] = num; sd[wid] = den; }
  __syncthreads();
  if (wid == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    num = lane < nw ? sn[lane] : 0.0;
    den = lane < nw ? sd[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      num += __shfl_xor_sync(0xffffffffu, num, o);
      den += __shfl_xor_sync(0xffffffffu, den, o);
    }
    if (lane == 0) {
      part[(((size_t)src * 6 + c) * 2 + 0) * kCheckBlocks + blockIdx.x] = num;
      part[(((size_t)src * 6 + c) * 2 + 1) * kCheckBlocks + blockIdx.x] = den;
    }
  }
}

// delta_g = sqrt(sum_g |now - prev|^2 / sum_g |now|^2) for g = E (components 0..2) and H (3..5); NaN where the
// denominator is 0 (nothing has reached the check set), as k_check_final reports it.  Components, then blocks, in order.
__global__ void k_check_final_static(const int nsrc, const int nblk, const double *__restrict__ part, double *__restrict__ delta) {
  const int src = blockIdx.x * blockDim.x + threadIdx.x;
  if (src >= nsrc) return;
  double sum[4] = {0.0, 0.0, 0.0, 0.0};
  for (int c = 0; c < 6; ++c)
    for (int q = 0; q < 2; ++q)
      for (int b = 0; b < nblk; ++b) sum[(c / 3) * 2 + q] += part[(((size_t)src * 6 + c) * 2 + q) * kCheckBlocks + b];
  delta[src * 2 + 0] = sum[1] > 0 ? sqrt(sum[0] / sum[1]) : nan("");
  delta[src * 2 + 1] = sum[3] > 0 ? sqrt(sum[2] / sum[3]) : nan("");
}

// device address of g_check_part on the current device; looked up on first use there (kMaxDev ordinals cached)
constexpr int kMaxDev = 64;
double *g_part_addr[kMaxDev] = {nullptr};

int static_scratch(double **out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(EMM_ECUDA, "emm_check_delta_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDev) return fail(EMM_EINVAL, "emm_check_delta_static: device ordinal %d beyond the %d this entry point keeps addresses for", dev, kMaxDev);
  if (!g_part_addr[dev]) {
    double *p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_check_part);
    if (e != cudaSuccess || !p) return fail(EMM_ECUDA, "emm_check_delta_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    g_part_addr[dev] = p;
  }
  *out = g_part_addr[dev];
  return 0;
}

}  // namespace

}  // namespace emm

using namespace emm;

extern "C" int emm_check_delta_static(const double *d_acc_now, const double *d_acc_prev, int nchk, int nsrc, double *d_delta, void *cuda_stream) {
  if (!d_acc_now || !d_acc_prev || !d_delta) return fail(EMM_EINVAL, "emm_check_delta_static: null argument");
  if (nsrc < 1 || nchk < 1) return fail(EMM_EINVAL, "emm_check_delta_static: nsrc and nchk must be >= 1");
  if (nsrc > kStaticMaxSrc)
    return fail(EMM_EINVAL, "emm_check_delta_static: %d sources exceed the static scratch, which holds the partial sums of at most %d (EMM_CHECK_STATIC_MAX_NSRC)",
                nsrc, kStaticMaxSrc);
  if (nchk > EMM_CHECK_STATIC_MAX_NCHK)
    return fail(EMM_EINVAL, "emm_check_delta_static: %d check-set points exceed the stated maximum of %d (EMM_CHECK_STATIC_MAX_NCHK)", nchk, EMM_CHECK_STATIC_MAX_NCHK);
  double *part = nullptr;
  int rc = static_scratch(&part);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int nb = (nchk + 255) / 256;                       // same block count rule as the run driver's check (launch_check)
  if (nb > kCheckBlocks) nb = kCheckBlocks;
  k_check_reduce_static<<<dim3(nb, 6, nsrc), 256, 0, st>>>(nchk, reinterpret_cast<const double2 *>(d_acc_now), reinterpret_cast<const double2 *>(d_acc_prev), part);
  k_check_final_static<<<(nsrc + 31) / 32, 32, 0, st>>>(nsrc, nb, part, d_delta);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(EMM_ECUDA, "emm_check_delta_static: %s", cudaGetErrorString(e));
  return 0;
}
