// S1: per-pad-row grid binning (BASELINE.json north_star; the paper, does not describe it).
// One CTA per (sector instance, pad row): counting sort of the row's clusters by z bin, done entirely in shared
// memory, writing the sorted (y,z) pairs, their original local indices and the bin-start table.
// The grid is an acceleration structure only; no result of S2..S6 depends on it.
#include "tpc_common.cuh"

namespace tpc {

constexpr int kBinThreads = 128;

__global__ void __launch_bounds__(kBinThreads)
bin_rows_kernel(const __grid_constant__ DevGeom g, const float4* __restrict__ clusters,
                const int32_t* __restrict__ row_offsets, float2* __restrict__ hit_yz, uint16_t* __restrict__ hit_idx,
                uint16_t* __restrict__ bin_start, int64_t* __restrict__ counts) {
    extern __shared__ uint32_t sm_hist[];  // [nz + 1] counts, then exclusive starts (running cursors in pass 2)
    __shared__ uint32_t sm_warp[kBinThreads / 32];
    const int slab = blockIdx.x;
    const int inst = slab / g.R;
    const int base = row_offsets[slab];
    int n = row_offsets[slab + 1] - base;
    if (n > 65535) {  // local indices are 16 bit: flag and ignore the excess (documented in tpc_tracker.h)
        if (threadIdx.x == 0) atomicOr((unsigned long long*)&counts[5], 1ull);
        n = 65535;
    }
    const float z0 = grid_z0(g, inst);
    const int nz = g.nz;
    for (int b = threadIdx.x; b <= nz; b += kBinThreads) sm_hist[b] = 0;
    __syncthreads();
    // pass 1: histogram.  Coalesced float4 loads, 16 B per thread.
    for (int i = threadIdx.x; i < n; i += kBinThreads) {
        const float4 c = __ldg(&clusters[base + i]);
        atomicAdd(&sm_hist[zbin(c.z, z0, g.inv_cz, nz)], 1u);
    }
    __syncthreads();
    // exclusive scan of nz+1 entries: contiguous chunk per thread, warp scan of the chunk sums
    const int per = (nz + 1 + kBinThreads - 1) / kBinThreads;
    const int lo = threadIdx.x * per, hi = min(lo + per, nz + 1);
    uint32_t sum = 0;
    for (int b = lo; b < hi; b++) sum += sm_hist[b];
    uint32_t incl = sum;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) sm_warp[wid] = incl;
    __syncthreads();
    uint32_t off = incl - sum;
    for (int k = 0; k < wid; k++) off += sm_warp[k];
    uint16_t* tbl = bin_start + (size_t)slab * g.nzp;
    for (int b = lo; b < hi; b++) {
        uint32_t c = sm_hist[b];
        sm_hist[b] = off;
        tbl[b] = (uint16_t)off;
        off += c;
    }
    __syncthreads();
    // pass 2: scatter (the clusters come from L1/L2 this time)
    for (int i = threadIdx.x; i < n; i += kBinThreads) {
        const float4 c = __ldg(&clusters[base + i]);
        const uint32_t pos = atomicAdd(&sm_hist[zbin(c.z, z0, g.inv_cz, nz)], 1u);
        hit_yz[base + pos] = make_float2(c.y, c.z);
        hit_idx[base + pos] = (uint16_t)i;
    }
}

int launch_bin_rows(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0) return 0;
    bin_rows_kernel<<<slabs, kBinThreads, (g.nz + 1) * sizeof(uint32_t), s>>>(
        g, p.clusters, p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start, w.counts);
    return 1;
}

}  // namespace tpc
