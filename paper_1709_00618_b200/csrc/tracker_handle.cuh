// The opaque handle behind tpc_tracker_t (private to the library's host code).
#pragma once
#include <string>

#include "../../include/tpc_tracker.h"
#include "tpc_common.cuh"

struct tpc_tracker {
    tpc::DevGeom g;
    float* d_row_x = nullptr;  // [3][R]: row_x, row_y0, row_inv_sy
    void* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    int n_sm = 148;
    int last_launches = 0;
    bool timing = false;
    bool input_yz = false;    // clusters are (y, z) pairs instead of (x, y, z, w) (tpc_set_input_layout)
    bool count_work = false;  // S5 work counters counts[6..9] (tpc_set_work_counters)
    cudaEvent_t ev[TPC_TIMING_RING][TPC_N_STAGES + 1] = {};
    bool ev_valid = false;
    int64_t n_calls = 0;  // timed calls so far (ring position = n_calls % TPC_TIMING_RING)
    std::string err;
};

static inline int fail(tpc_tracker* t, int code, const std::string& msg) {
    if (t) t->err = msg;
    return code;
}

