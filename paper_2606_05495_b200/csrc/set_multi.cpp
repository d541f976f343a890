// set_multi.cpp -- several scheduler instances behind one submit call (include/set.h "set_multi_*").
// Built on the public C ABI only: an instance is a whole set_ctx (own streams, slots, executables, dispatcher) on the device
// it was given.  A job's home is job_id mod n; an instance that has room takes a job whose home has none -- host-side
// stealing across instances at the moment of submission, before anything was bound to an executable, so the steal costs
// nothing but the scan (the paper's retarget-to-thief, rebinding an already prepared graph, is what a steal
// INSIDE an instance does).  No collective and no device-to-device traffic: the jobs live in host memory.
#include <atomic>
#include <vector>

#include "set.h"

struct set_multi {
    std::vector<set_ctx*> inst;
    std::atomic<uint64_t> stolen{0};
};

extern "C" {

set_status set_multi_destroy(set_multi* m) {
    if (!m) return SET_OK;
    set_status first = SET_OK;
    for (set_ctx* c : m->inst) {
        set_status rc = set_destroy(c);
        if (first == SET_OK) first = rc;
    }
    delete m;
    return first;
}

set_status set_multi_create(const set_config* cfg, int num_instances, const int* devices, set_multi** out) {
    if (out) *out = nullptr;
    if (!cfg || !devices || !out || num_instances < 1 || num_instances > 64) return SET_ERR_INVALID;
    if (cfg->mode != SET_MODE_SET) return SET_ERR_INVALID;
    set_multi* m = new set_multi;
    for (int i = 0; i < num_instances; ++i) {
        set_config c = *cfg;
        c.device = devices[i];
        set_ctx* ctx = nullptr;
        set_status rc = set_create_ex(&c, &ctx);
        if (rc != SET_OK) {
            set_multi_destroy(m);
            return rc;
        }
        m->inst.push_back(ctx);
    }
    *out = m;
    return SET_OK;
}

set_status set_multi_register_pipeline(set_multi* m, const set_stage_desc* stages, int num_stages, const set_buffer_desc* bufs, int num_bufs) {
    if (!m) return SET_ERR_INVALID;
    for (set_ctx* c : m->inst)
        if (set_status rc = set_register_pipeline(c, stages, num_stages, bufs, num_bufs)) return rc;
    return SET_OK;
}

set_status set_multi_submit_dims(set_multi* m, uint64_t job_id, const void* host_in, void* host_out, const uint32_t dims[SET_MAX_DIMS]) {
    if (!m || m->inst.empty()) return SET_ERR_INVALID;
    const size_t n = m->inst.size(), home = (size_t)(job_id % n);
    for (size_t k = 0; k < n; ++k) {  // home first, then home + 1, home + 2, ... cyclically
        size_t i = home + k;
        if (i >= n) i -= n;
        set_status rc = set_try_submit_dims(m->inst[i], job_id, host_in, host_out, dims);
        if (rc == SET_OK) {
            if (k) m->stolen.fetch_add(1, std::memory_order_relaxed);
            return SET_OK;
        }
        if (rc != SET_ERR_BUSY) return rc;
    }
    return set_submit_dims(m->inst[home], job_id, host_in, host_out, dims);  // every instance is full: back-pressure at home
}

set_status set_multi_drain(set_multi* m) {
    if (!m) return SET_ERR_INVALID;
    set_status first = SET_OK;
    for (set_ctx* c : m->inst) {
        set_status rc = set_drain(c);
        if (first == SET_OK) first = rc;
    }
    return first;
}

set_ctx* set_multi_instance(set_multi* m, int i) { return (m && i >= 0 && (size_t)i < m->inst.size()) ? m->inst[(size_t)i] : nullptr; }

uint64_t set_multi_stolen(set_multi* m) { return m ? m->stolen.load(std::memory_order_relaxed) : 0; }

}  // extern "C"
