// detect.cuh -- the thresholded candidate list over the block maxima (reading 20; "detect").
//
// The hot kernel in OUT_BLOCKMAX mode leaves, per (batch item, template row, block of S columns), the maximum
// power and the lowest column offset attaining it (reading 17).  These three small kernels turn that into the
// list a search pipeline wants: every block maximum >= threshold (float32, inclusive) as (item, row, column,
// power), ordered by (item, row, column), at most `capacity` of them, with the count of all of them.
// The arrays are n_batch * n_z * n_blk entries (C3: 235 371; C5: 3.2 M): a few microseconds of HBM/L2 traffic
// next to the milliseconds of the correlation, so clarity and determinism come first: count per row, scan,
// ordered scatter.  No atomics: the position of a candidate depends only on the data.
#pragma once
#include <stdint.h>

#include "../../include/fdas.h"

namespace fdas {

// one warp per (item, row): how many of its block maxima pass the threshold
__global__ void __launch_bounds__(256) fdas_cand_count_kernel(const float *__restrict__ bmax, int n_rows, long long n_blk,
                                                              float thr, int *__restrict__ row_count)
{
    const int w = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (w >= n_rows) return;
    const float *b = bmax + (long long)w * n_blk;
    int c = 0;
    for (long long s0 = lane; s0 < n_blk; s0 += 128) { // four independent loads in flight per lane
        float v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = (s0 + 32 * u < n_blk) ? b[s0 + 32 * u] : -1.f;
#pragma unroll
        for (int u = 0; u < 4; ++u) c += (s0 + 32 * u < n_blk && v[u] >= thr) ? 1 : 0;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    if (lane == 0) row_count[w] = c;
}

// one CTA: row_count[0 .. n_rows) -> exclusive prefix sums in place, row_count[n_rows] = total;
// d_count[0] = total (all candidates), d_count[1] = min(total, capacity) (candidates written)
__global__ void __launch_bounds__(1024) fdas_cand_scan_kernel(int *__restrict__ row_count, int n_rows, int capacity,
                                                              int *__restrict__ d_count)
{
    __shared__ int part[1024];
    const int t = threadIdx.x;
    const int per = (n_rows + 1023) / 1024;
    const int r0 = min(n_rows, t * per), r1 = min(n_rows, r0 + per);
    int s = 0;
    for (int r = r0; r < r1; ++r) s += row_count[r];
    part[t] = s;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) { // inclusive scan of the per-thread sums
        const int v = (t >= d) ? part[t - d] : 0;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    int run = part[t] - s; // exclusive prefix of this thread's chunk
    for (int r = r0; r < r1; ++r) {
        const int c = row_count[r];
        row_count[r] = run;
        run += c;
    }
    if (t == 1023) {
        const int total = part[1023];
        row_count[n_rows] = total;
        d_count[0] = total;
        d_count[1] = total < capacity ? total : capacity;
    }
}

// one warp per (item, row): its candidates, in column order, to their places in the list
__global__ void __launch_bounds__(256) fdas_cand_scatter_kernel(const float *__restrict__ bmax, const int *__restrict__ barg,
                                                                int n_rows, int n_z, long long n_blk, int blk, float thr,
                                                                const int *__restrict__ row_offset, int capacity,
                                                                fdas_candidate *__restrict__ cand)
{
    const int w = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (w >= n_rows) return;
    int base = row_offset[w];
    if (base >= capacity) return; // the list is already full before this row
    const float *b = bmax + (long long)w * n_blk;
    const int *a = barg + (long long)w * n_blk;
    const int row_end = row_offset[w + 1];   // one past this row's last place: nothing left to find beyond it
    for (long long s0 = 0; s0 < n_blk && base < capacity && base < row_end; s0 += 128) {
        float v[4];                           // four independent loads in flight per lane, consumed in column order
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const long long s = s0 + 32 * u + lane;
            v[u] = s < n_blk ? b[s] : 0.f;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const long long s = s0 + 32 * u + lane;
            const bool hit = s < n_blk && v[u] >= thr;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            const int pos = base + __popc(m & ((1u << lane) - 1u));
            if (hit && pos < capacity) {
                fdas_candidate c;
                c.item = w / n_z;
                c.row = w % n_z;
                c.column = (int32_t)(s * blk + a[s]);
                c.power = v[u];
                cand[pos] = c;
            }
            base += __popc(m);
        }
    }
}

} // namespace fdas
