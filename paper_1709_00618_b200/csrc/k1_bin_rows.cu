// S1: per-pad-row grid binning (BASELINE.json north_star; the paper, does not describe it).
// One CTA per (sector instance, pad row): counting sort of the row's clusters by grid cell (z bin major, y strip
// minor), done entirely in shared memory, writing the sorted (y,z) pairs, their original local indices and the
// cell-start table.  The grid is an acceleration structure only; no result of S2..S6 depends on it.
#include <mutex>

#include "tpc_common.cuh"

namespace tpc {

constexpr int kBinThreads = 128;

#ifndef TPC_BIN_CTAS
#define TPC_BIN_CTAS 16
#endif
// (y, z) of input cluster i in one of the three input layouts (tpc_set_input_layout): (x, y, z, w) records, compact
// (y, z) pairs, or 16-bit fixed point (y = q_y / 256 cm; z = z origin of the sector side + q_z / 64 cm, q_z unsigned).
// The fixed-point decode is one exact multiplication and, for z, one rounded addition (exact for origins that are
// multiples of 1/64 cm and |z| < 2^18 / 64): the oracle's input is produced by the same two operations on the host.
enum InLayout : int { kInXYZW = 0, kInYZ = 1, kInI16 = 2 };

template <int kIn>
__device__ __forceinline__ float2 load_yz(const void* __restrict__ in, int i, float z_origin) {
    if (kIn == kInYZ) return __ldg(reinterpret_cast<const float2*>(in) + i);
    if (kIn == kInI16) {
        const short2 q = __ldg(reinterpret_cast<const short2*>(in) + i);
        return make_float2(__fmul_rn((float)q.x, 1.0f / 256.0f),
                           __fadd_rn(z_origin, __fmul_rn((float)(unsigned short)q.y, 1.0f / 64.0f)));
    }
    const float4 c = __ldg(reinterpret_cast<const float4*>(in) + i);
    return make_float2(c.y, c.z);
}

template <int kIn>
__global__ void __launch_bounds__(kBinThreads, TPC_BIN_CTAS)
bin_rows_kernel(const __grid_constant__ DevGeom g, const void* __restrict__ clusters,
                const int32_t* __restrict__ row_offsets, float2* __restrict__ hit_yz, uint16_t* __restrict__ hit_idx,
                uint16_t* __restrict__ hit_pos, uint16_t* __restrict__ bin_start, int64_t* __restrict__ counts) {
    // Cell counters are 16 bit, two per 32-bit word (a row holds <= 65,535 hits, so neither half can carry into the
    // other): half the shared memory, half the zeroing and half the scan work of 32-bit counters, and the scanned
    // words ARE the uint16 cell table that goes to global memory.
    extern __shared__ __align__(16) uint32_t sm_hist[];  // [nzp / 2] packed counts, then exclusive starts (cursors)
    __shared__ uint32_t sm_warp[kBinThreads / 32];
    const int slab = blockIdx.x;
    const int inst = slab / g.R, r = slab - inst * g.R;
    const int base = row_offsets[slab];
    int n = row_offsets[slab + 1] - base;
    if (n > 65535) {  // local indices are 16 bit: flag and ignore the excess (documented in tpc_tracker.h)
        if (threadIdx.x == 0) atomicOr((unsigned long long*)&counts[5], 1ull);
        n = 65535;
    }
    const float z0 = grid_z0(g, inst);
    const float y0 = g.row_y0[r], inv_sy = g.row_inv_sy[r];
    const int nw = g.nzp / 2;  // packed words; nzp % 16 == 0, so nw % 8 == 0
    uint4* hist4 = reinterpret_cast<uint4*>(sm_hist);
    for (int b = threadIdx.x; b < nw / 4; b += kBinThreads) hist4[b] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    // pass 1: histogram.  Coalesced loads; the cell ids stay in registers for pass 2 when the row is short enough
    // (two hits per thread), which is the normal case.
    constexpr int kKeep = 2;
    int key[kKeep];
    float2 yz[kKeep];
#pragma unroll
    for (int k = 0; k < kKeep; k++) {
        const int i = threadIdx.x + k * kBinThreads;
        key[k] = -1;
        if (i < n) {
            const float2 c = load_yz<kIn>(clusters, base + i, z0);
            key[k] = zbin(c.y, z0, g.inv_cz, g.nz) * g.ny + ybin(c.x, y0, inv_sy, g.ny);
            yz[k] = c;
            atomicAdd(&sm_hist[key[k] >> 1], (key[k] & 1) ? 0x10000u : 1u);
        }
    }
    for (int i = threadIdx.x + kKeep * kBinThreads; i < n; i += kBinThreads) {
        const float2 c = load_yz<kIn>(clusters, base + i, z0);
        const int kk = zbin(c.y, z0, g.inv_cz, g.nz) * g.ny + ybin(c.x, y0, inv_sy, g.ny);
        atomicAdd(&sm_hist[kk >> 1], (kk & 1) ? 0x10000u : 1u);
    }
    __syncthreads();
    // exclusive scan of the nzp counters: a contiguous chunk of 4-word groups (8 cells) per thread, warp scan of the
    // chunk sums
    const int groups = nw / 4;
    const int per = (groups + kBinThreads - 1) / kBinThreads;
    const int glo = min(threadIdx.x * per, groups), ghi = min(glo + per, groups);
    uint32_t sum = 0;
    for (int q = glo; q < ghi; q++) {
        const uint4 a = hist4[q];
        const uint32_t t = a.x + a.y + a.z + a.w;  // sums of the low and of the high halves, each <= 65,535
        sum += (t & 0xffffu) + (t >> 16);
    }
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
    uint4* tbl4 = reinterpret_cast<uint4*>(bin_start + (size_t)slab * g.nzp);  // 16-B aligned: nzp % 8 == 0
    for (int q = glo; q < ghi; q++) {
        const uint4 a = hist4[q];
        uint4 o;
        uint32_t lo, hi;
        lo = a.x & 0xffffu; hi = a.x >> 16; o.x = off | ((off + lo) << 16); off += lo + hi;
        lo = a.y & 0xffffu; hi = a.y >> 16; o.y = off | ((off + lo) << 16); off += lo + hi;
        lo = a.z & 0xffffu; hi = a.z >> 16; o.z = off | ((off + lo) << 16); off += lo + hi;
        lo = a.w & 0xffffu; hi = a.w >> 16; o.w = off | ((off + lo) << 16); off += lo + hi;
        hist4[q] = o;
        tbl4[q] = o;
    }
    __syncthreads();
    // pass 2: scatter (the packed start of a cell is its cursor: atomicAdd returns the word before the increment)
#pragma unroll
    for (int k = 0; k < kKeep; k++) {
        if (key[k] >= 0) {
            const uint32_t w = atomicAdd(&sm_hist[key[k] >> 1], (key[k] & 1) ? 0x10000u : 1u);
            const uint32_t pos = (key[k] & 1) ? (w >> 16) : (w & 0xffffu);
            hit_yz[base + pos] = yz[k];
            hit_idx[base + pos] = (uint16_t)(threadIdx.x + k * kBinThreads);
            hit_pos[base + threadIdx.x + k * kBinThreads] = (uint16_t)pos;  // inverse permutation, coalesced
        }
    }
    for (int i = threadIdx.x + kKeep * kBinThreads; i < n; i += kBinThreads) {  // long rows: from L1/L2 this time
        const float2 c = load_yz<kIn>(clusters, base + i, z0);
        const int kk = zbin(c.y, z0, g.inv_cz, g.nz) * g.ny + ybin(c.x, y0, inv_sy, g.ny);
        const uint32_t w = atomicAdd(&sm_hist[kk >> 1], (kk & 1) ? 0x10000u : 1u);
        const uint32_t pos = (kk & 1) ? (w >> 16) : (w & 0xffffu);
        hit_yz[base + pos] = c;
        hit_idx[base + pos] = (uint16_t)i;
        hit_pos[base + i] = (uint16_t)pos;
    }
}

int launch_bin_rows(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0) return 0;
    const size_t smem = (size_t)g.nzp * sizeof(uint16_t);
    if (smem > 48 * 1024) {  // opt-in size, a property of (kernel, device): cached per device ordinal
        static std::mutex mu;
        static size_t configured[kMaxDeviceOrdinals] = {};
        int dev = 0;
        cudaGetDevice(&dev);
        dev = dev >= 0 && dev < kMaxDeviceOrdinals ? dev : 0;
        std::lock_guard<std::mutex> lock(mu);
        if (smem > configured[dev]) {
            cudaFuncSetAttribute(bin_rows_kernel<kInXYZW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(bin_rows_kernel<kInYZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(bin_rows_kernel<kInI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            configured[dev] = smem;
        }
    }
    if (p.layout == kInYZ)
        bin_rows_kernel<kInYZ><<<slabs, kBinThreads, smem, s>>>(g, p.clusters, p.row_offsets, w.hit_yz, w.hit_idx,
                                                                w.hit_pos, w.bin_start, w.counts);
    else if (p.layout == kInI16)
        bin_rows_kernel<kInI16><<<slabs, kBinThreads, smem, s>>>(g, p.clusters, p.row_offsets, w.hit_yz, w.hit_idx,
                                                                 w.hit_pos, w.bin_start, w.counts);
    else
        bin_rows_kernel<kInXYZW><<<slabs, kBinThreads, smem, s>>>(g, p.clusters, p.row_offsets, w.hit_yz, w.hit_idx,
                                                                  w.hit_pos, w.bin_start, w.counts);
    return 1;
}

}  // namespace tpc
