// dc_blank.cuh -- the blanking logic that consumes direct cuts: union of holes and AB faces,
// Algorithm 3.1 steps 6-7 (L121-L125).  Pure label arithmetic: one thread per element, streaming (HBM bound:
// 3-4 bytes per element in, 1 out), lists by warp-aggregated atomic append.
#pragma once

__global__ void k_union_labels(long long n, const signed char *__restrict__ a, const signed char *__restrict__ b, signed char *out)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int x = a[e], y = b[e];
    out[e] = (signed char)((x == DC_HOLE || y == DC_HOLE) ? DC_HOLE : ((x == DC_CUT || y == DC_CUT) ? DC_CUT : DC_NORMAL));
}

__device__ __forceinline__ void warp_append(bool mine, int id, int *list, long long cap, unsigned long long *counter)
{
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    if (!m) return;
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(counter, (unsigned long long)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (mine && list) {
        const unsigned long long pos = base + __popc(m & ((1u << lane) - 1));
        if (pos < (unsigned long long)cap) list[pos] = id;
    }
}

__global__ void k_unblank(int mode, int cut_is_hole, long long n, const signed char *__restrict__ prev,
                          const signed char *__restrict__ lt, const signed char *__restrict__ lp, signed char *out,
                          int *unblank_list, int *tohole_list, long long cap, unsigned long long *counts)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    bool unb = false, toh = false;
    if (e < n) {
        const int a = lt[e], b = lp[e];
        const bool was = prev[e] != 0;
        const bool ht = a == DC_HOLE || (cut_is_hole && a == DC_CUT);
        const bool hp = b == DC_HOLE || (cut_is_hole && b == DC_CUT);
        // wall: 6.1 hole at t or t+dt -> hole, 6.2 unblank if hole in neither; overset: hole only if hole in both, 7.1
        const bool blank = mode == DC_MODE_WALL ? (ht || hp) : (ht && hp);
        unb = was && !blank;
        toh = blank && !was;
        out[e] = blank ? 1 : 0;
    }
    warp_append(unb, (int)e, unblank_list, cap, counts);
    warp_append(toh, (int)e, tohole_list, cap, counts + 1);
}

__global__ void k_ab_faces(long long n, const signed char *__restrict__ ib, const int *__restrict__ adj,
                           unsigned char *__restrict__ mask, unsigned long long *count)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int m = 0;
    if (e < n && ib[e] == 0) {
        const int2 *ap = reinterpret_cast<const int2 *>(adj + e * 6);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int2 v = __ldg(ap + k);
            if (v.x >= 0 && ib[v.x] != 0) m |= 1 << (2 * k);
            if (v.y >= 0 && ib[v.y] != 0) m |= 1 << (2 * k + 1);
        }
    }
    if (e < n) mask[e] = (unsigned char)m;
    if (count) {
        int c = __popc(m);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, (unsigned long long)c);
    }
}

extern "C" int dc_union_labels(long long n_elem, const signed char *a_dev, const signed char *b_dev, signed char *out_dev, void *stream)
{
    if (n_elem <= 0 || !a_dev || !b_dev || !out_dev) return DC_ERR_ARG;
    k_union_labels<<<nblk(n_elem, 256), 256, 0, (cudaStream_t)stream>>>(n_elem, a_dev, b_dev, out_dev);
    CK(cudaGetLastError());
    return DC_OK;
}

extern "C" int dc_unblank(int mode, int cut_is_hole, long long n_elem, const signed char *iblank_prev_dev,
                          const signed char *labels_t_dev, const signed char *labels_tplus_dev, signed char *iblank_out_dev,
                          int *unblank_list_dev, int *tohole_list_dev, long long list_cap, long long *counts_dev, void *stream)
{
    if (n_elem <= 0 || !iblank_prev_dev || !labels_t_dev || !labels_tplus_dev || !iblank_out_dev || !unblank_list_dev ||
        !counts_dev || list_cap < 0 || (mode != DC_MODE_WALL && mode != DC_MODE_OVERSET)) return DC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemsetAsync(counts_dev, 0, 16, st));
    k_unblank<<<nblk(n_elem, 256), 256, 0, st>>>(mode, cut_is_hole, n_elem, iblank_prev_dev, labels_t_dev, labels_tplus_dev,
                                                 iblank_out_dev, unblank_list_dev, tohole_list_dev, list_cap,
                                                 reinterpret_cast<unsigned long long *>(counts_dev));
    CK(cudaGetLastError());
    return DC_OK;
}

extern "C" int dc_ab_faces(long long n_elem, const signed char *iblank_dev, const int *adj6_dev, unsigned char *ab_mask_dev,
                           long long *count_dev, void *stream)
{
    if (n_elem <= 0 || !iblank_dev || !adj6_dev || !ab_mask_dev) return DC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (count_dev) CK(cudaMemsetAsync(count_dev, 0, 8, st));
    k_ab_faces<<<nblk(n_elem, 256), 256, 0, st>>>(n_elem, iblank_dev, adj6_dev, ab_mask_dev, reinterpret_cast<unsigned long long *>(count_dev));
    CK(cudaGetLastError());
    return DC_OK;
}
