// noalloc.cu -- nanobte_get_boundary_heat_noalloc: the boundary heat per tag (O8; PAPER.md:51, 129 -- the heat that
// leaves through the faces of one boundary tag) for callers that may not allocate (code under CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  A variant of tagheat_kernel (kernels_common.cu): there one block
// walks all faces of a tag and the per-tag sums go through a device buffer of the solver's arena; here the faces of a tag
// are split over kNoallocChunks blocks, whose partial sums go through a STATIC device array, and a second kernel joins
// them in a fixed order.  Nothing is allocated, by this file or by anything it calls.
//
// The scratch array is part of the library image: every GPU that loads libnanobte.so holds its 34 KiB until the process
// exits.  In host code its name is a host-side stand-in, not a device address; the address comes from
// cudaGetSymbolAddress, once per device, with that device current (scratch_for_current_device below).
// Every call on a device shares the array, and it keeps the last call's contents: both kernels overwrite every entry they
// later read (a block with no faces writes 0), so nothing has to be cleared -- but two calls that overlap on one GPU
// (different streams, different solvers) race on it.
#include <mutex>

#include "internal.h"

namespace {

constexpr int kNoallocMaxTags = NANOBTE_NOALLOC_MAX_TAGS;  // 256
constexpr int kNoallocChunks = 16;                         // blocks per tag
constexpr int kNoallocMaxDevices = 64;

// [kNoallocMaxTags][kNoallocChunks] partial sums, then [kNoallocMaxTags] joined sums (staging for a host destination)
static __device__ __align__(256) double g_tagheat_scratch[kNoallocMaxTags * (kNoallocChunks + 1)];

// [tag][chunk] partial sums: chunk c of tag t takes the faces k = lo + c*256 + thread, stepping kNoallocChunks*256.
__global__ void __launch_bounds__(256) tagheat_split_kernel(const int32_t *tagface_ptr, const int32_t *tagface,
                                                            const double *faceflux, const double *bf_area, int B,
                                                            double *scratch) {
  __shared__ double red[256];
  const int t = blockIdx.y, c = blockIdx.x;
  double acc = 0.0;
  for (int k = tagface_ptr[t] + c * 256 + threadIdx.x; k < tagface_ptr[t + 1]; k += kNoallocChunks * 256) {
    const int bf = tagface[k];
    double F = 0.0;
    for (int b = 0; b < B; ++b) F += faceflux[(size_t)bf * B + b];
    acc += bf_area[bf] * F;
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) scratch[t * kNoallocChunks + c] = red[0];
}

__global__ void tagheat_join_kernel(int n_tags, const double *scratch, double *out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_tags) return;
  double acc = 0.0;
  for (int c = 0; c < kNoallocChunks; ++c) acc += scratch[t * kNoallocChunks + c];
  out[t] = acc;
}

// Device address of g_tagheat_scratch on the current device: looked up once per device and remembered.
int scratch_for_current_device(nanobte_solver *h, double **out) {
  static std::mutex mu;
  static double *addr[kNoallocMaxDevices] = {};
  int dev = -1;
  NB_CUDA(h, cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoallocMaxDevices) return nb_fail(h, NANOBTE_E_INVALID, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    double *p = nullptr;
    NB_CUDA(h, cudaGetSymbolAddress((void **)&p, g_tagheat_scratch));
    if (!p) return nb_fail(h, NANOBTE_E_CUDA, "cudaGetSymbolAddress gave no address for the static scratch");
    addr[dev] = p;
  }
  *out = addr[dev];
  return 0;
}

}  // namespace

extern "C" int nanobte_get_boundary_heat_noalloc(nanobte_solver *h, double *per_tag, int32_t dst_is_device) {
  if (!h || !h->arena || !per_tag) return NANOBTE_E_INVALID;
  if (h->n_tags > kNoallocMaxTags)
    return nb_fail(h, NANOBTE_E_INVALID,
                   "nanobte_get_boundary_heat_noalloc: %d boundary tags, the static scratch holds at most %d "
                   "(NANOBTE_NOALLOC_MAX_TAGS); use nanobte_get_boundary_heat",
                   h->n_tags, kNoallocMaxTags);
  if (h->n_tags == 0) return 0;
  double *scratch = nullptr;
  int rc = scratch_for_current_device(h, &scratch);
  if (rc < 0) return rc;
  rc = nb_refresh_thermalizing(h);  // as nanobte_get_boundary_heat does: kernels only
  if (rc < 0) return rc;
  tagheat_split_kernel<<<dim3(kNoallocChunks, h->n_tags), 256, 0, h->stream>>>(h->tagface_ptr, h->tagface, h->bd.faceflux,
                                                                              h->bd.bf_area, h->B, scratch);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  double *stage = scratch + kNoallocMaxTags * kNoallocChunks;  // host destination: staged in the scratch's tail
  double *out = dst_is_device ? per_tag : stage;
  tagheat_join_kernel<<<(h->n_tags + 127) / 128, 128, 0, h->stream>>>(h->n_tags, scratch, out);
  h->launches++;
  NB_CUDA(h, cudaGetLastError());
  if (!dst_is_device) {
    NB_CUDA(h, cudaMemcpyAsync(per_tag, stage, (size_t)h->n_tags * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    NB_CUDA(h, cudaStreamSynchronize(h->stream));
  }
  return 0;
}
