// stream.cu -- the step before the hot path for a continuous stream (reading F):
//   corner turn   telescope blocks are time-major ([t][chan], SIGPROC order) and may have the lowest frequency first;
//                 the search wants channel-major rows with the highest frequency first ("frequency flip")
//   overlap-save  aamulti reads each segment with an overlap so that every DM trial has its full sweep:
//                 the working buffer keeps the last `history` samples of every channel row and appends the new block.
// Both are pure data movement, HBM bound.
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

// out[b][c'][t0 + t] = in[b][t][c],  c' = flip ? nchan-1-c : c.  Tile: 64 samples x 128 channels through shared memory;
// loads are 128-byte rows of channels, stores are 64-byte runs of samples.
// The input is addressed as in[b*in_beam_stride + t*in_t_stride + c]: a block per beam ([beam][t][chan]: strides nsamp*nchan
// and nchan) or time-spliced over the beams ([t][beam][chan]: strides nchan and nbeam*nchan).
__global__ void __launch_bounds__(256) corner_turn_kernel(const uint8_t* __restrict__ in, int64_t nsamp, int32_t nchan,
                                                          int64_t in_beam_stride, int64_t in_t_stride,
                                                          int32_t flip, uint8_t* __restrict__ out, int64_t out_row_stride,
                                                          int64_t out_beam_stride, int64_t out_t0) {
    __shared__ uint8_t tile[128][64 + 4];                 // [channel][sample], padded rows
    const int b = blockIdx.z;
    const int64_t t0 = (int64_t)blockIdx.x * 64;
    const int c0 = blockIdx.y * 128;
    const uint8_t* src = in + (int64_t)b * in_beam_stride;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;          // 32 x 8
    // load: one warp reads 128 consecutive channels of one sample (4 per lane)
    for (int i = ty; i < 64; i += 8) {
        const int64_t t = t0 + i;
        const int c = c0 + 4 * tx;
        uint32_t v = 0;
        if (t < nsamp) {
            const uint8_t* p = src + t * in_t_stride + c;
            if (c + 4 <= nchan && ((reinterpret_cast<uintptr_t>(p) & 3) == 0)) v = *reinterpret_cast<const uint32_t*>(p);
            else
                for (int k = 0; k < 4; ++k)
                    if (c + k < nchan) v |= (uint32_t)p[k] << (8 * k);
        }
        tile[4 * tx + 0][i] = (uint8_t)v;
        tile[4 * tx + 1][i] = (uint8_t)(v >> 8);
        tile[4 * tx + 2][i] = (uint8_t)(v >> 16);
        tile[4 * tx + 3][i] = (uint8_t)(v >> 24);
    }
    __syncthreads();
    // store: 16 lanes write the 64 samples of one channel (4 per lane), two channels per warp pass
    const int half = tx >> 4, l = tx & 15;
    for (int i = ty * 2 + half; i < 128; i += 16) {
        const int c = c0 + i;
        if (c >= nchan) continue;
        const int cc = flip ? nchan - 1 - c : c;
        const int64_t t = t0 + 4 * l;
        uint8_t* dst = out + (int64_t)b * out_beam_stride + (int64_t)cc * out_row_stride + out_t0 + t;
        const uint32_t v = *reinterpret_cast<const uint32_t*>(&tile[i][4 * l]);
        if (t + 4 <= nsamp && ((reinterpret_cast<uintptr_t>(dst) & 3) == 0)) *reinterpret_cast<uint32_t*>(dst) = v;
        else
            for (int k = 0; k < 4; ++k)
                if (t + k < nsamp) dst[k] = (uint8_t)(v >> (8 * k));
    }
}

// The same for the aligned case (4 | nchan, 4 | every stride and offset, 4-byte aligned pointers), which is what telescope
// blocks are: tile = 128 samples x 128 channels.  A thread loads a 4 x 4 micro-tile (four 32-bit words: 4 channels of 4
// consecutive samples), transposes it in registers with byte permutes and stores four words -- 4 samples of one channel each --
// into a swizzled shared tile (word column tq of channel c at c*32 + (tq ^ (c >> 2)): stores and loads are both conflict free);
// then every warp writes whole 128-byte runs of samples per channel.  All global accesses are 128-byte warp transactions.
__global__ void __launch_bounds__(256) corner_turn_fast_kernel(const uint8_t* __restrict__ in, int64_t nsamp, int32_t nchan,
                                                               int64_t in_beam_stride, int64_t in_t_stride, int32_t flip,
                                                               uint8_t* __restrict__ out, int64_t out_row_stride,
                                                               int64_t out_beam_stride, int64_t out_t0) {
    __shared__ uint32_t tile[128 * 32];                    // [channel][sample quad], swizzled
    const int b = blockIdx.z;
    const int64_t t0 = (int64_t)blockIdx.x * 128;
    const int c0 = blockIdx.y * 128;
    const uint8_t* src = in + (int64_t)b * in_beam_stride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c = c0 + 4 * lane;                           // this lane's four channels
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int tq = warp + 8 * it;                      // sample quad of the tile
        const int64_t t = t0 + 4 * tq;
        uint32_t r[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            r[j] = (c < nchan && t + j < nsamp) ? __ldg(reinterpret_cast<const uint32_t*>(src + (t + j) * in_t_stride + c)) : 0u;
        const uint32_t a = __byte_perm(r[0], r[1], 0x5140), bq = __byte_perm(r[2], r[3], 0x5140);
        const uint32_t cq = __byte_perm(r[0], r[1], 0x7362), d = __byte_perm(r[2], r[3], 0x7362);
        const int col = tq ^ lane;                         // (4*lane + i) >> 2 == lane
        tile[(4 * lane + 0) * 32 + col] = __byte_perm(a, bq, 0x5410);
        tile[(4 * lane + 1) * 32 + col] = __byte_perm(a, bq, 0x7632);
        tile[(4 * lane + 2) * 32 + col] = __byte_perm(cq, d, 0x5410);
        tile[(4 * lane + 3) * 32 + col] = __byte_perm(cq, d, 0x7632);
    }
    __syncthreads();
#pragma unroll 4
    for (int i = warp; i < 128; i += 8) {                  // one channel row per warp pass: 32 lanes x 4 samples = 128 bytes
        const int ch = c0 + i;
        if (ch >= nchan) break;
        const int64_t t = t0 + 4 * lane;
        if (t >= nsamp) continue;
        const uint32_t v = tile[i * 32 + (lane ^ (i >> 2))];
        const int cc = flip ? nchan - 1 - ch : ch;
        uint8_t* dst = out + (int64_t)b * out_beam_stride + (int64_t)cc * out_row_stride + out_t0 + t;
        if (t + 4 <= nsamp) *reinterpret_cast<uint32_t*>(dst) = v;
        else
            for (int k = 0; k < 4; ++k)
                if (t + k < nsamp) dst[k] = (uint8_t)(v >> (8 * k));
    }
}

void launch_corner_turn(const uint8_t* in, int32_t nbeam, int64_t nsamp, int32_t nchan, int32_t flip, int32_t spliced,
                        uint8_t* out, int64_t out_row_stride, int64_t out_beam_stride, int64_t out_t0, cudaStream_t st) {
    if (nbeam <= 0 || nsamp <= 0 || nchan <= 0) return;
    {
        const int64_t beam_stride = spliced ? (int64_t)nchan : nsamp * (int64_t)nchan;
        const int64_t t_stride = spliced ? (int64_t)nbeam * nchan : (int64_t)nchan;
        const bool aligned = (nchan & 3) == 0 && (out_row_stride & 3) == 0 && (out_beam_stride & 3) == 0 && (out_t0 & 3) == 0 &&
                             (reinterpret_cast<uintptr_t>(in) & 3) == 0 && (reinterpret_cast<uintptr_t>(out) & 3) == 0;
        if (aligned) {
            dim3 grid((unsigned)((nsamp + 127) / 128), (unsigned)((nchan + 127) / 128), (unsigned)nbeam);
            corner_turn_fast_kernel<<<grid, 256, 0, st>>>(in, nsamp, nchan, beam_stride, t_stride, flip, out, out_row_stride,
                                                          out_beam_stride, out_t0);
            return;
        }
    }
    dim3 grid((unsigned)((nsamp + 63) / 64), (unsigned)((nchan + 127) / 128), (unsigned)nbeam);
    const int64_t beam_stride = spliced ? (int64_t)nchan : nsamp * (int64_t)nchan;
    const int64_t t_stride = spliced ? (int64_t)nbeam * nchan : (int64_t)nchan;
    corner_turn_kernel<<<grid, 256, 0, st>>>(in, nsamp, nchan, beam_stride, t_stride, flip, out, out_row_stride, out_beam_stride,
                                             out_t0);
}

// dst[row][0 .. nkeep) = src[row][shift .. shift + nkeep): the history of every channel row moves to the front of the
// other working buffer (all counts are multiples of 16 bytes).
__global__ void keep_history_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, int64_t row16, int64_t shift16,
                                    int64_t keep16, int64_t nrows) {
    const int64_t n = keep16 * nrows;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / keep16, k = i - r * keep16;
        dst[r * row16 + k] = __ldg(src + r * row16 + shift16 + k);
    }
}

void launch_keep_history(const uint8_t* src, uint8_t* dst, int64_t row_bytes, int64_t shift_bytes, int64_t keep_bytes,
                         int64_t nrows, cudaStream_t st) {
    if (keep_bytes <= 0 || nrows <= 0) return;
    keep_history_kernel<<<sm_count() * 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(src), reinterpret_cast<uint4*>(dst),
                                                  row_bytes / 16, shift_bytes / 16, keep_bytes / 16, nrows);
}

}  // namespace spt
