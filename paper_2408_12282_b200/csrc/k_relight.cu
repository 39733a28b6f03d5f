// Relighting from a precomputed reflectance field (second half; "To speed up
// generation we can precompute a reflectance field assuming white light.  We compute the relit view as the sum over
// the reflectance field scaled by the environment illumination."):
//     out[p][c] = sum_l weights[l][c] * frames[l][p][c]
// over the OLAT frames [L][P][3] of one view.  Pure streaming work: 12 (L + 1) P bytes, two flops per 4 bytes read --
// the HBM roofline bounds it, there is nothing for the tensor cores here.
//
// Layout of the work: a frame is a flat array of 3 P floats.  A warp owns 96 consecutive float4 (384 floats = 128
// pixels, a multiple of 3 so that the colour phase of a float4 depends on the lane only) and reads them as three
// fully coalesced 512-byte rows per light; each lane keeps three float4 accumulators and picks the weight of each
// of its 12 elements once per light with selects (element e of the frame has channel e mod 3).  Lights are unrolled
// by four, so 12 independent 16-byte loads per thread are in flight; loads and stores bypass L1 allocation
// (read-once / write-once data).  Frames whose float count is not a multiple of 4 (P % 4 != 0: later frames are
// not 16-byte aligned) take the scalar kernel.
#include "internal.cuh"

namespace sssgs {

namespace {

__device__ __forceinline__ float4 ld_stream(const float4* p) { return __ldcs(p); }

__global__ void __launch_bounds__(256)
relight_vec_kernel(const float4* __restrict__ frames, int n_light, int64_t frame_stride4, const float* __restrict__ weights,
                   float4* __restrict__ out, int64_t n4) {
  const int lane = threadIdx.x & 31;
  const int64_t warps_total = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t n_units = (n4 + 95) / 96;
  // channel of the first element of this lane's float4 in row m: (lane + 32 m) mod 3 (the unit's base is a multiple of 3)
  int ph[3];
#pragma unroll
  for (int m = 0; m < 3; ++m) ph[m] = (lane + 2 * m) % 3;
  for (int64_t u = (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5); u < n_units; u += warps_total) {
    const int64_t j0 = u * 96 + lane;
    float4 acc[3];
    bool ok[3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      acc[m] = make_float4(0.f, 0.f, 0.f, 0.f);
      ok[m] = j0 + 32 * m < n4;
    }
#pragma unroll 4
    for (int l = 0; l < n_light; ++l) {
      const float4* f = frames + (int64_t)l * frame_stride4 + j0;
      float4 x[3];
#pragma unroll
      for (int m = 0; m < 3; ++m) x[m] = ok[m] ? ld_stream(f + 32 * m) : make_float4(0.f, 0.f, 0.f, 0.f);
      const float wr = __ldg(weights + 3 * l), wg = __ldg(weights + 3 * l + 1), wb = __ldg(weights + 3 * l + 2);
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const float w0 = ph[m] == 0 ? wr : (ph[m] == 1 ? wg : wb);
        const float w1 = ph[m] == 0 ? wg : (ph[m] == 1 ? wb : wr);
        const float w2 = ph[m] == 0 ? wb : (ph[m] == 1 ? wr : wg);
        acc[m].x = fmaf(w0, x[m].x, acc[m].x);
        acc[m].y = fmaf(w1, x[m].y, acc[m].y);
        acc[m].z = fmaf(w2, x[m].z, acc[m].z);
        acc[m].w = fmaf(w0, x[m].w, acc[m].w);
      }
    }
#pragma unroll
    for (int m = 0; m < 3; ++m)
      if (ok[m]) __stcs(out + j0 + 32 * m, acc[m]);
  }
}

__global__ void __launch_bounds__(256)
relight_scalar_kernel(const float* __restrict__ frames, int n_light, int64_t frame_stride, const float* __restrict__ weights,
                      float* __restrict__ out, int64_t n) {
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    const int c = (int)(e % 3);
    float acc = 0.f;
    for (int l = 0; l < n_light; ++l) acc = fmaf(__ldg(weights + 3 * l + c), __ldcs(frames + (int64_t)l * frame_stride + e), acc);
    __stcs(out + e, acc);
  }
}

}  // namespace

int launch_relight(const float* frames, int n_light, int64_t n_pixels, const float* weights, float* out, int num_sms,
                   cudaStream_t s) {
  const int64_t n = n_pixels * 3;
  if (n == 0) return 0;
  if ((n_pixels & 3) == 0) {
    const int64_t n4 = n / 4;
    const int64_t units = (n4 + 95) / 96;
    int64_t blocks = (units + 7) / 8;                       // 8 warps per CTA, one unit per warp and trip
    const int64_t cap = (int64_t)num_sms * 8;               // 8 resident CTAs of 256 threads per SM
    if (blocks > cap) blocks = cap;
    relight_vec_kernel<<<(unsigned)blocks, 256, 0, s>>>(reinterpret_cast<const float4*>(frames), n_light, n4,
                                                        weights, reinterpret_cast<float4*>(out), n4);
  } else {
    int64_t blocks = (n + 255) / 256;
    const int64_t cap = (int64_t)num_sms * 8;
    if (blocks > cap) blocks = cap;
    relight_scalar_kernel<<<(unsigned)blocks, 256, 0, s>>>(frames, n_light, n, weights, out, n);
  }
  return 1;
}

}  // namespace sssgs
