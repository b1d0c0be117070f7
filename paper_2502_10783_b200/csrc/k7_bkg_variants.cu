// K7: the pixel-level piece of the background variants: growing the detections of one iteration and
// joining them with the caller's bad-pixel mask (readings B4, B5; "We will iterate to remove background noises
// with the background estimation and removal function").  out = (bad0 != 0) | dilate(det, grow), the dilation by the
// (2 grow + 1)^2 square clipped at the frame edge.  A byte-mask stencil: 1 B/px read (+1 B/px for bad0), 1 B/px written;
// one thread per 4 pixels, three aligned 32-bit loads per window row turned into a 12-bit "non-zero" mask.
#include "common.cuh"

namespace {

__device__ __forceinline__ uint32_t nz_nibble(uint32_t v) {   // 4 bytes -> 4 bits (byte != 0)
    const uint32_t nz = ((((v & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | v) & 0x80808080u) >> 7;
    return (nz * 0x00204081u >> 21) & 0xFu;
}

__global__ void __launch_bounds__(256) k7_dilate_or_kernel(const uint8_t *det, const uint8_t *bad0, int H, int W, int grow,
                                                           uint8_t *out) {
    const int w4 = W >> 2;
    const int x4 = blockIdx.x * blockDim.x + threadIdx.x;
    const int frame = blockIdx.z;
    if (x4 >= w4) return;
    const size_t fbase = (size_t)frame * H * W;
  for (int y = blockIdx.y; y < H; y += gridDim.y) {   // gridDim.y = min(H, 65535): one row per block unless the frame is taller
    uint32_t any = 0;   // bit q: pixel 4 x4 + q has a detection in its window
    if (det) {
        const int y0 = max(y - grow, 0), y1 = min(y + grow, H - 1);
        const uint32_t wmask = (1u << (2 * grow + 1)) - 1u;
        for (int yy = y0; yy <= y1; ++yy) {
            const uint32_t *row = reinterpret_cast<const uint32_t *>(det + fbase + (size_t)yy * W);
            const uint32_t l = x4 > 0 ? __ldg(row + x4 - 1) : 0u, m = __ldg(row + x4), r = x4 + 1 < w4 ? __ldg(row + x4 + 1) : 0u;
            const uint32_t m12 = nz_nibble(l) | nz_nibble(m) << 4 | nz_nibble(r) << 8;   // bit k: byte 4 (x4 - 1) + k != 0
#pragma unroll
            for (int q = 0; q < 4; ++q) any |= (((m12 >> (4 + q - grow)) & wmask) ? 1u : 0u) << q;
        }
    }
    uint32_t o = (any & 1u) | (any & 2u) << 7 | (any & 4u) << 14 | (any & 8u) << 21;
    if (bad0) {
        const uint32_t b = __ldg(reinterpret_cast<const uint32_t *>(bad0 + fbase + (size_t)y * W) + x4);
        const uint32_t nb = nz_nibble(b);
        o |= (nb & 1u) | (nb & 2u) << 7 | (nb & 4u) << 14 | (nb & 8u) << 21;
    }
    reinterpret_cast<uint32_t *>(out + fbase + (size_t)y * W)[x4] = o;
  }
}

}  // namespace

int k7_dilate_or(bd_ctx *ctx, const uint8_t *d_det, const uint8_t *d_bad0, int B, int H, int W, int grow, uint8_t *d_out,
                 cudaStream_t st) {
    dim3 grid((W / 4 + 255) / 256, H < 65535 ? H : 65535, B);
    k7_dilate_or_kernel<<<grid, 256, 0, st>>>(d_det, d_bad0, H, W, grow, d_out);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
