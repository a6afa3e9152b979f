// Host-buffer entry points (include/tpc_tracker.h): tpc_pipeline_create / run / destroy and the one-shot
// tpc_track_sectors_host.  BASELINE.json configs[4]: drift windows "streamed through the tracker in double-buffered
// chunks with cluster upload overlapped on a second CUDA stream"; PAPER.md:100 (time frames are sliced when they do
// not fit); PAPER.md:33 names the host<->GPU transfer as the bottleneck of this kind of offload.
//
// Streams: one for uploads, one for downloads, and one compute stream per slot that has its own workspace (else a
// single shared one).  Chunk i+1 uploads while chunk i is tracked and the results of earlier chunks go back; with
// per-slot workspaces the first stages of chunk i+1 also fill the SMs that the drain phase of chunk i's follower
// leaves idle.  The host thread only waits for the 128-byte counts of a chunk whose successors are already queued, so
// the GPU never idles on it.  Everything the pipeline needs besides the caller's buffers (streams, events, a pinned
// counts buffer) is created once in tpc_pipeline_create: a run allocates nothing.
#include <chrono>
#include <new>
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

}  // namespace

struct tpc_pipeline {
    tpc_tracker* t = nullptr;
    std::vector<tpc_slot_t> slots;
    bool own_streams = false;
    bool per_slot_ws = false;  // every slot has its own workspace -> its own compute stream
    cudaStream_t s_in = nullptr, s_out = nullptr;
    std::vector<cudaStream_t> s_cmp;  // per slot (all equal when the workspace is shared)
    // per slot: start / end of the upload, the tracking and the download of the chunk that uses it
    std::vector<cudaEvent_t> in0, in1, cmp0, cmp1, out0, out1;
    int64_t* h_counts = nullptr;  // pinned [n_slots][TPC_N_COUNTS]
};

static void destroy_pipeline(tpc_pipeline* p) {
    if (!p) return;
    for (auto* v : {&p->in0, &p->in1, &p->cmp0, &p->cmp1, &p->out0, &p->out1})
        for (cudaEvent_t e : *v)
            if (e) cudaEventDestroy(e);
    if (p->own_streams) {
        if (p->s_in) cudaStreamDestroy(p->s_in);
        if (p->s_out) cudaStreamDestroy(p->s_out);
        for (size_t i = 0; i < p->s_cmp.size(); i++)
            if (p->s_cmp[i] && (i == 0 || p->s_cmp[i] != p->s_cmp[0])) cudaStreamDestroy(p->s_cmp[i]);
    }
    if (p->h_counts) cudaFreeHost(p->h_counts);
    delete p;
}

// streams == nullptr: the pipeline creates its own (non-blocking); else {h2d, compute, d2h} of the caller
static int make_pipeline(tpc_tracker* t, const tpc_slot_t* slots, int32_t n_slots, cudaStream_t* streams,
                         tpc_pipeline** out) {
    if (!t) return TPC_ERR_ARG;
    if (!slots || !out || n_slots < 2 || n_slots > 8) return fail(t, TPC_ERR_ARG, "2..8 slots are required");
    *out = nullptr;
    bool all_ws = true;
    for (int s = 0; s < n_slots; s++) {
        if (!slots[s].clusters || !slots[s].row_offsets || !slots[s].out.counts || slots[s].max_clusters < 0 ||
            slots[s].max_instances < 1)
            return fail(t, TPC_ERR_ARG, "slot buffers missing");
        if (slots[s].workspace && ((uintptr_t)slots[s].workspace & 255))
            return fail(t, TPC_ERR_ARG, "slot workspace must be 256-byte aligned");
        all_ws = all_ws && slots[s].workspace != nullptr;
    }
    tpc_pipeline* p = new (std::nothrow) tpc_pipeline();
    if (!p) return fail(t, TPC_ERR_ARG, "out of host memory");
    p->t = t;
    p->slots.assign(slots, slots + n_slots);
    p->per_slot_ws = all_ws && streams == nullptr;
    p->own_streams = streams == nullptr;
    p->s_cmp.assign(n_slots, nullptr);
    cudaError_t e = cudaSuccess;
    if (streams) {
        p->s_in = streams[0];
        p->s_out = streams[2];
        for (int s = 0; s < n_slots; s++) p->s_cmp[s] = streams[1];
    } else {
        e = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking);
        for (int s = 0; s < n_slots && e == cudaSuccess; s++) {
            if (s == 0 || p->per_slot_ws)
                e = cudaStreamCreateWithFlags(&p->s_cmp[s], cudaStreamNonBlocking);
            else
                p->s_cmp[s] = p->s_cmp[0];
        }
    }
    for (auto* v : {&p->in0, &p->in1, &p->cmp0, &p->cmp1, &p->out0, &p->out1}) {
        v->assign(n_slots, nullptr);
        for (int s = 0; s < n_slots && e == cudaSuccess; s++) e = cudaEventCreate(&(*v)[s]);
    }
    if (e == cudaSuccess) e = cudaHostAlloc(&p->h_counts, sizeof(int64_t) * TPC_N_COUNTS * n_slots, cudaHostAllocDefault);
    if (e != cudaSuccess) {
        destroy_pipeline(p);
        return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
    }
    *out = p;
    return TPC_OK;
}

extern "C" int tpc_pipeline_create(tpc_tracker_t* t, const tpc_slot_t* slots, int32_t n_slots, tpc_pipeline_t** out) {
    return make_pipeline(t, slots, n_slots, nullptr, out);
}

extern "C" void tpc_pipeline_destroy(tpc_pipeline_t* p) { destroy_pipeline(p); }

#define CK(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            rc = fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e_)); \
            goto done;                                                                   \
        }                                                                                \
    } while (0)

extern "C" int tpc_pipeline_run(tpc_pipeline_t* p, const void* h_cl_v, const int32_t* h_ro, int32_t n_inst,
                                int64_t n_clusters, int32_t inst_per_chunk, tpc_host_output_t* hout) {
    if (!p) return TPC_ERR_ARG;
    tpc_tracker* t = p->t;
    if (!h_ro || !hout || inst_per_chunk < 1 || n_inst < 0 || n_clusters < 0) return fail(t, TPC_ERR_ARG, "bad argument");
    if (n_clusters > 0 && !h_cl_v) return fail(t, TPC_ERR_ARG, "NULL clusters");
    // the chunks run on the slots' workspaces and streams: whatever an earlier tpc_track_sectors call left for
    // tpc_merge_refit is stale from here on (phase 2 needs a tpc_track_sectors call of its own)
    t->last_ws = nullptr;
    const auto wall0 = std::chrono::steady_clock::now();
    const int R = t->g.R;
    const int n_slots = (int)p->slots.size();
    const int64_t bpc = layout_bytes(t->input_layout);  // bytes per cluster in h_clusters and in the slots
    const char* h_cl = static_cast<const char*>(h_cl_v);
    std::vector<Chunk> chunks;
    for (int32_t i0 = 0; i0 < n_inst; i0 += inst_per_chunk) {
        Chunk c;
        c.inst0 = i0;
        c.n_inst = (n_inst - i0 < inst_per_chunk) ? n_inst - i0 : inst_per_chunk;
        c.cl0 = h_ro[(int64_t)i0 * R];
        c.n_cl = h_ro[(int64_t)(i0 + c.n_inst) * R] - c.cl0;
        chunks.push_back(c);
    }
    for (const tpc_slot_t& sl : p->slots)
        for (const Chunk& c : chunks)
            if (c.n_cl > sl.max_clusters || c.n_inst > sl.max_instances)
                return fail(t, TPC_ERR_ARG, "a chunk exceeds the slot capacity");
    int rc = TPC_OK;
    const int nc = (int)chunks.size();
    int64_t launches = 0, up_bytes = 0, down_bytes = 0;
    int64_t track_base = 0, hit_base = 0;
    double ms_in = 0.0, ms_cmp = 0.0, ms_out = 0.0;
    for (int i = 0; i < TPC_N_COUNTS; i++) hout->totals[i] = 0;
    cudaStream_t s_in = p->s_in, s_out = p->s_out;

    // completes chunk j: wait for its counts, make indices job-wide, send the results home
    auto finish = [&](int j) -> int {
        const int s = j % n_slots;
        const Chunk& c = chunks[j];
        cudaError_t e = cudaEventSynchronize(p->cmp1[s]);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p->in0[s], p->in1[s]);
        ms_in += ms;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p->cmp0[s], p->cmp1[s]);
        ms_cmp += ms;
        if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
        const int64_t* cnt = p->h_counts + (size_t)s * TPC_N_COUNTS;
        const tpc_output_t& o = p->slots[s].out;
        int64_t nt = cnt[3], nh = cnt[4];
        if (nt > o.trk_capacity) nt = o.trk_capacity;
        if (o.trk_hits && nh > o.trk_hits_capacity) nh = o.trk_hits_capacity;
        for (int i = 0; i < TPC_N_COUNTS; i++)
            hout->totals[i] = (i == 5) ? (hout->totals[i] | cnt[i]) : hout->totals[i] + cnt[i];
        int ret = TPC_OK;
        if (cnt[3] > o.trk_capacity || (o.trk_hits && cnt[4] > o.trk_hits_capacity))
            ret = fail(t, TPC_ERR_CAPACITY, "slot track capacity too small");
        // The job-wide host arrays are full: this chunk (and every later one) is not downloaded, but its slot still
        // gets an (empty) download interval and the bases advance, so that the run goes on to the end and
        // hout->totals report the sizes the caller needs.
        const bool host_full =
            track_base + nt > hout->trk_capacity || (hout->trk_hits && hit_base + nh > hout->trk_hits_capacity);
        if (host_full) ret = fail(t, TPC_ERR_CAPACITY, "host track capacity too small");
        e = cudaEventRecord(p->out0[s], s_out);
        if (c.n_cl > 0 && e == cudaSuccess && !host_full) {
            int32_t* d_owner = (hout->cluster_owner && o.cluster_owner) ? o.cluster_owner : nullptr;
            int32_t* d_hits = (hout->trk_hits && o.trk_hits) ? o.trk_hits : nullptr;
            int64_t* d_off = (hout->trk_hit_offset && o.trk_hit_offset) ? o.trk_hit_offset : nullptr;
            int32_t* d_sec = (hout->trk_sector && o.trk_sector) ? o.trk_sector : nullptr;
            if (d_owner || d_hits || d_off || d_sec) {
                globalise_kernel<<<t->n_sm * 4, 256, 0, s_out>>>(d_owner, c.n_cl, (int32_t)track_base, d_hits, nh,
                                                                 (int32_t)c.cl0, d_off, d_sec, nt, hit_base, c.inst0);
                e = cudaGetLastError();
                launches++;
            }
            auto back = [&](void* dst, const void* src, size_t bytes) {
                if (dst && src && bytes && e == cudaSuccess) {
                    e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s_out);
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
        if (e == cudaSuccess) e = cudaEventRecord(p->out1[s], s_out);
        if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
        return ret;
    };
    // the download interval of the chunk that used slot s last (read before its events are recorded again)
    auto read_out_ms = [&](int s) -> cudaError_t {
        cudaError_t e = cudaEventSynchronize(p->out1[s]);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p->out0[s], p->out1[s]);
        ms_out += ms;
        return e;
    };

    for (int i = 0; i < nc; i++) {
        const int s = i % n_slots;
        const Chunk& c = chunks[i];
        const tpc_slot_t& sl = p->slots[s];
        cudaStream_t s_cmp = p->s_cmp[s];
        if (i >= 2 * n_slots) CK(read_out_ms(s));
        if (i >= n_slots) {
            const int r = finish(i - n_slots);
            if (r == TPC_ERR_CAPACITY) rc = r;  // keep going (also after the first one): the totals tell the required sizes
            else if (r != TPC_OK) { rc = r; goto done; }
        }
        // upload: the slot's inputs are free once the chunk that used them last has been tracked
        if (i >= n_slots) CK(cudaStreamWaitEvent(s_in, p->cmp1[s], 0));
        CK(cudaEventRecord(p->in0[s], s_in));
        if (c.n_cl > 0) {
            CK(cudaMemcpyAsync(sl.clusters, h_cl + bpc * c.cl0, (size_t)(bpc * c.n_cl), cudaMemcpyHostToDevice, s_in));
            up_bytes += bpc * c.n_cl;
        }
        const int64_t n_ro = (int64_t)c.n_inst * R + 1;
        CK(cudaMemcpyAsync(sl.row_offsets, h_ro + (int64_t)c.inst0 * R, sizeof(int32_t) * n_ro, cudaMemcpyHostToDevice, s_in));
        up_bytes += (int64_t)sizeof(int32_t) * n_ro;
        CK(cudaEventRecord(p->in1[s], s_in));
        // track: needs the upload, and the slot's outputs must have left (chunk i - n_slots)
        CK(cudaStreamWaitEvent(s_cmp, p->in1[s], 0));
        if (i >= n_slots) CK(cudaStreamWaitEvent(s_cmp, p->out1[s], 0));
        CK(cudaEventRecord(p->cmp0[s], s_cmp));
        if (c.cl0 != 0) {
            rebase_offsets_kernel<<<64, 256, 0, s_cmp>>>(sl.row_offsets, n_ro);
            zero_first_kernel<<<1, 1, 0, s_cmp>>>(sl.row_offsets);
            CK(cudaGetLastError());
            launches += 2;
        }
        {
            void* ws = p->per_slot_ws ? sl.workspace : t->ws;
            const size_t wsb = p->per_slot_ws ? sl.workspace_bytes : t->ws_bytes;
            const int r = tpc_track_on(t, ws, wsb, s_cmp, false, c.inst0, sl.clusters, sl.row_offsets, c.n_inst, c.n_cl, &sl.out);
            if (r != TPC_OK) { rc = r; goto done; }
            launches += t->last_launches;
        }
        CK(cudaMemcpyAsync(p->h_counts + (size_t)s * TPC_N_COUNTS, sl.out.counts, sizeof(int64_t) * TPC_N_COUNTS,
                           cudaMemcpyDeviceToHost, s_cmp));
        down_bytes += (int64_t)sizeof(int64_t) * TPC_N_COUNTS;
        CK(cudaEventRecord(p->cmp1[s], s_cmp));
    }
    for (int j = (nc > n_slots ? nc - n_slots : 0); j < nc; j++) {
        if (j >= n_slots) CK(read_out_ms(j % n_slots));
        const int r = finish(j);
        if (r == TPC_ERR_CAPACITY) rc = r;
        else if (r != TPC_OK) { rc = r; goto done; }
    }
    for (int j = (nc > n_slots ? nc - n_slots : 0); j < nc; j++) CK(read_out_ms(j % n_slots));
    if (hout->trk_hit_offset && track_base <= hout->trk_capacity) hout->trk_hit_offset[track_base] = hit_base;
    CK(cudaStreamSynchronize(s_out));
done:
    if (rc != TPC_OK) {  // drain whatever is in flight before the caller's buffers go away
        cudaStreamSynchronize(s_in);
        for (cudaStream_t s : p->s_cmp) cudaStreamSynchronize(s);
        cudaStreamSynchronize(s_out);
    }
    hout->n_chunks = nc;
    hout->n_launches = launches;
    hout->h2d_bytes = up_bytes;
    hout->d2h_bytes = down_bytes;
    hout->h2d_ms = (float)ms_in;
    hout->compute_ms = (float)ms_cmp;
    hout->d2h_ms = (float)ms_out;
    hout->wall_ms = std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - wall0).count();
    return rc;
}

extern "C" int tpc_track_sectors_host(tpc_tracker_t* t, const void* h_cl, const int32_t* h_ro, int32_t n_inst,
                                      int64_t n_clusters, int32_t inst_per_chunk, tpc_slot_t* slots, int32_t n_slots,
                                      void* h2d_stream, void* compute_stream, void* d2h_stream,
                                      tpc_host_output_t* hout) {
    cudaStream_t streams[3] = {static_cast<cudaStream_t>(h2d_stream), static_cast<cudaStream_t>(compute_stream),
                               static_cast<cudaStream_t>(d2h_stream)};
    tpc_pipeline* p = nullptr;
    int rc = make_pipeline(t, slots, n_slots, streams, &p);
    if (rc != TPC_OK) return rc;
    rc = tpc_pipeline_run(p, h_cl, h_ro, n_inst, n_clusters, inst_per_chunk, hout);
    destroy_pipeline(p);
    return rc;
}
