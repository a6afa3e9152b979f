// tpc_track_sectors_host: the host-buffer entry point (include/tpc_tracker.h).  BASELINE.json configs[4]: drift
// windows "streamed through the tracker in double-buffered chunks with cluster upload overlapped on a second CUDA
// stream"; PAPER.md:100 (time frames are sliced when they do not fit).  Three streams: chunk i+1 uploads while chunk
// i is tracked and the results of chunk i-1 go back.  The host thread only waits for the 128-byte counts of a chunk
// whose successor is already queued, so the GPU never idles on it.
#include <vector>

#include "tracker_handle.cuh"

using namespace tpc;

namespace {

__global__ void rebase_offsets_kernel(int32_t* __restrict__ ro, int64_t n) {
    // chunk row offsets arrive with the job-wide base; make them start at 0 (device-side, no host pass over them)
    const int32_t base = ro[0];
    __shared__ int32_t s_base;
    if (threadIdx.x == 0) s_base = base;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x + 1; i < n; i += (int64_t)gridDim.x * blockDim.x)
        ro[i] -= s_base;
}

__global__ void zero_first_kernel(int32_t* ro) { ro[0] = 0; }

// make the chunk-local indices job-wide before they leave the device
__global__ void globalise_kernel(int32_t* __restrict__ owner, int64_t n_clusters, int32_t track_base,
                                 int32_t* __restrict__ trk_hits, int64_t n_hits, int32_t cluster_base,
                                 int64_t* __restrict__ hit_offset, int32_t* __restrict__ trk_sector, int64_t n_tracks,
                                 int64_t hit_base, int32_t inst_base) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (owner)
        for (int64_t i = t0; i < n_clusters; i += stride) {
            const int32_t o = owner[i];
            if (o >= 0) owner[i] = o + track_base;
        }
    if (trk_hits)
        for (int64_t i = t0; i < n_hits; i += stride) trk_hits[i] += cluster_base;
    if (hit_offset)
        for (int64_t i = t0; i < n_tracks; i += stride) hit_offset[i] += hit_base;
    if (trk_sector)
        for (int64_t i = t0; i < n_tracks; i += stride) trk_sector[i] += inst_base;
}

struct Chunk {
    int32_t inst0, n_inst;
    int64_t cl0, n_cl;
};

#define CK(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            rc = fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e_)); \
            goto done;                                                                   \
        }                                                                                \
    } while (0)

}  // namespace

extern "C" int tpc_track_sectors_host(tpc_tracker_t* t, const float* h_cl, const int32_t* h_ro, int32_t n_inst,
                                      int64_t n_clusters, int32_t inst_per_chunk, tpc_slot_t* slots, int32_t n_slots,
                                      void* h2d_stream, void* compute_stream, void* d2h_stream,
                                      tpc_host_output_t* hout) {
    if (!t) return TPC_ERR_ARG;
    if (!h_ro || !slots || !hout || n_slots < 2 || n_slots > 8 || inst_per_chunk < 1 || n_inst < 0 || n_clusters < 0)
        return fail(t, TPC_ERR_ARG, "bad argument");
    if (n_clusters > 0 && !h_cl) return fail(t, TPC_ERR_ARG, "NULL clusters");
    const int R = t->g.R;
    const int64_t fpc = t->input_yz ? 2 : 4;  // floats per cluster in h_cl and in the slots' cluster buffers
    cudaStream_t s_in = static_cast<cudaStream_t>(h2d_stream), s_cmp = static_cast<cudaStream_t>(compute_stream),
                 s_out = static_cast<cudaStream_t>(d2h_stream);
    std::vector<Chunk> chunks;
    for (int32_t i0 = 0; i0 < n_inst; i0 += inst_per_chunk) {
        Chunk c;
        c.inst0 = i0;
        c.n_inst = (n_inst - i0 < inst_per_chunk) ? n_inst - i0 : inst_per_chunk;
        c.cl0 = h_ro[(int64_t)i0 * R];
        c.n_cl = h_ro[(int64_t)(i0 + c.n_inst) * R] - c.cl0;
        chunks.push_back(c);
    }
    for (int s = 0; s < n_slots; s++) {
        if (!slots[s].clusters || !slots[s].row_offsets || !slots[s].out.counts)
            return fail(t, TPC_ERR_ARG, "slot buffers missing");
        for (const Chunk& c : chunks)
            if (c.n_cl > slots[s].max_clusters || c.n_inst > slots[s].max_instances)
                return fail(t, TPC_ERR_ARG, "a chunk exceeds the slot capacity");
    }
    int rc = TPC_OK;
    const int nc = (int)chunks.size();
    std::vector<cudaEvent_t> ev_in(n_slots), ev_cmp(n_slots), ev_out(n_slots);
    int64_t* h_counts = nullptr;  // pinned [n_slots][TPC_N_COUNTS]
    int64_t launches = 0, up_bytes = 0, down_bytes = 0;
    int64_t track_base = 0, hit_base = 0;
    for (int i = 0; i < TPC_N_COUNTS; i++) hout->totals[i] = 0;
    cudaStream_t saved_stream = t->stream;
    bool ev_made = false;

    // completes chunk j: wait for its counts, make indices job-wide, send the results home
    auto finish = [&](int j) -> int {
        const int s = j % n_slots;
        const Chunk& c = chunks[j];
        cudaError_t e = cudaEventSynchronize(ev_cmp[s]);
        if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
        const int64_t* cnt = h_counts + (size_t)s * TPC_N_COUNTS;
        const tpc_output_t& o = slots[s].out;
        int64_t nt = cnt[3], nh = cnt[4];
        if (nt > o.trk_capacity) nt = o.trk_capacity;
        if (nh > o.trk_hits_capacity) nh = o.trk_hits_capacity;
        for (int i = 0; i < TPC_N_COUNTS; i++) hout->totals[i] = (i == 5) ? (hout->totals[i] | cnt[i]) : hout->totals[i] + cnt[i];
        if (cnt[3] > o.trk_capacity || cnt[4] > o.trk_hits_capacity) rc = fail(t, TPC_ERR_CAPACITY, "slot track capacity too small");
        if (track_base + nt > hout->trk_capacity || hit_base + nh > hout->trk_hits_capacity)
            return fail(t, TPC_ERR_CAPACITY, "host track capacity too small");
        if (c.n_cl > 0) {
            const bool need_fix = (o.cluster_owner && hout->cluster_owner) || (o.trk_hits && hout->trk_hits) ||
                                  (o.trk_hit_offset && hout->trk_hit_offset) || (o.trk_sector && hout->trk_sector);
            if (need_fix) {
                globalise_kernel<<<t->n_sm * 4, 256, 0, s_out>>>(
                    hout->cluster_owner ? o.cluster_owner : nullptr, c.n_cl, (int32_t)track_base,
                    hout->trk_hits ? o.trk_hits : nullptr, nh, (int32_t)c.cl0,
                    hout->trk_hit_offset ? o.trk_hit_offset : nullptr, hout->trk_sector ? o.trk_sector : nullptr, nt,
                    hit_base, c.inst0);
                launches++;
            }
            auto back = [&](void* dst, const void* src, size_t bytes) {
                if (dst && src && bytes) {
                    cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s_out);
                    down_bytes += (int64_t)bytes;
                }
            };
            back(hout->cluster_owner ? hout->cluster_owner + c.cl0 : nullptr, o.cluster_owner, sizeof(int32_t) * c.n_cl);
            back(hout->trk_hits ? hout->trk_hits + hit_base : nullptr, o.trk_hits, sizeof(int32_t) * nh);
            back(hout->trk_params ? hout->trk_params + track_base * 5 : nullptr, o.trk_params, sizeof(float) * 5 * nt);
            back(hout->trk_cov ? hout->trk_cov + track_base * 15 : nullptr, o.trk_cov, sizeof(float) * 15 * nt);
            back(hout->trk_nhits ? hout->trk_nhits + track_base : nullptr, o.trk_nhits, sizeof(int32_t) * nt);
            back(hout->trk_sector ? hout->trk_sector + track_base : nullptr, o.trk_sector, sizeof(int32_t) * nt);
            back(hout->trk_hit_offset ? hout->trk_hit_offset + track_base : nullptr, o.trk_hit_offset, sizeof(int64_t) * nt);
        }
        track_base += nt;
        hit_base += nh;
        e = cudaEventRecord(ev_out[s], s_out);
        if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
        return TPC_OK;
    };

    CK(cudaHostAlloc(&h_counts, sizeof(int64_t) * TPC_N_COUNTS * n_slots, cudaHostAllocDefault));
    for (int s = 0; s < n_slots; s++) {
        CK(cudaEventCreateWithFlags(&ev_in[s], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ev_cmp[s], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ev_out[s], cudaEventDisableTiming));
    }
    ev_made = true;
    t->stream = s_cmp;
    for (int i = 0; i < nc; i++) {
        const int s = i % n_slots;
        const Chunk& c = chunks[i];
        if (i >= n_slots) {
            const int r = finish(i - n_slots);
            if (r != TPC_OK) { rc = r; goto done; }
        }
        // upload: the slot's inputs are free once the chunk that used them last has been tracked
        if (i >= n_slots) CK(cudaStreamWaitEvent(s_in, ev_cmp[s], 0));
        if (c.n_cl > 0) {
            // TPC_INPUT_YZ: 2 floats per cluster instead of 4 (tpc_set_input_layout)
            CK(cudaMemcpyAsync(slots[s].clusters, h_cl + fpc * c.cl0, sizeof(float) * fpc * c.n_cl, cudaMemcpyHostToDevice, s_in));
            up_bytes += (int64_t)sizeof(float) * fpc * c.n_cl;
        }
        const int64_t n_ro = (int64_t)c.n_inst * R + 1;
        CK(cudaMemcpyAsync(slots[s].row_offsets, h_ro + (int64_t)c.inst0 * R, sizeof(int32_t) * n_ro, cudaMemcpyHostToDevice, s_in));
        up_bytes += (int64_t)sizeof(int32_t) * n_ro;
        CK(cudaEventRecord(ev_in[s], s_in));
        // track: needs the upload, and the slot's outputs must have left (chunk i - n_slots)
        CK(cudaStreamWaitEvent(s_cmp, ev_in[s], 0));
        if (i >= n_slots) CK(cudaStreamWaitEvent(s_cmp, ev_out[s], 0));
        if (c.cl0 != 0) {
            rebase_offsets_kernel<<<64, 256, 0, s_cmp>>>(slots[s].row_offsets, n_ro);
            zero_first_kernel<<<1, 1, 0, s_cmp>>>(slots[s].row_offsets);
            launches += 2;
        }
        {
            const int r = tpc_track_sectors(t, slots[s].clusters, slots[s].row_offsets, c.n_inst, c.n_cl, &slots[s].out);
            if (r != TPC_OK) { rc = r; goto done; }
            launches += t->last_launches;
        }
        CK(cudaMemcpyAsync(h_counts + (size_t)s * TPC_N_COUNTS, slots[s].out.counts, sizeof(int64_t) * TPC_N_COUNTS,
                           cudaMemcpyDeviceToHost, s_cmp));
        down_bytes += (int64_t)sizeof(int64_t) * TPC_N_COUNTS;
        CK(cudaEventRecord(ev_cmp[s], s_cmp));
    }
    for (int j = (nc > n_slots ? nc - n_slots : 0); j < nc; j++) {
        const int r = finish(j);
        if (r != TPC_OK) { rc = r; goto done; }
    }
    if (hout->trk_hit_offset && track_base <= hout->trk_capacity) hout->trk_hit_offset[track_base] = hit_base;
    CK(cudaStreamSynchronize(s_out));
done:
    if (rc != TPC_OK) {  // drain whatever is in flight before the buffers go away
        cudaStreamSynchronize(s_in);
        cudaStreamSynchronize(s_cmp);
        cudaStreamSynchronize(s_out);
    }
    t->stream = saved_stream;
    if (ev_made)
        for (int s = 0; s < n_slots; s++) {
            cudaEventDestroy(ev_in[s]);
            cudaEventDestroy(ev_cmp[s]);
            cudaEventDestroy(ev_out[s]);
        }
    if (h_counts) cudaFreeHost(h_counts);
    hout->n_chunks = nc;
    hout->n_launches = launches;
    hout->h2d_bytes = up_bytes;
    hout->d2h_bytes = down_bytes;
    return rc;
}
