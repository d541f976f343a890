// set_trace.cpp -- libsettrace: device-timeline gaps from CUPTI activity records (include/set_trace.h).
// Measurement infrastructure of SURVEY.md §8(d) "Gaps"; not on the dispatch path and not linked into libset.so.
// libcupti is dlopen'ed on first use so that the host-only reduction (set_trace_reduce) works on a CPU-only box.
#include <dlfcn.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include <cupti.h>

#include "../../include/set_trace.h"

namespace {

std::string g_err;
std::mutex g_mu;
std::vector<set_trace_rec> g_recs;
uint64_t g_dropped = 0;
bool g_on = false;

struct Cupti {
    void* h = nullptr;
    CUptiResult (*RegisterCallbacks)(CUpti_BuffersCallbackRequestFunc, CUpti_BuffersCallbackCompleteFunc) = nullptr;
    CUptiResult (*Enable)(CUpti_ActivityKind) = nullptr;
    CUptiResult (*Disable)(CUpti_ActivityKind) = nullptr;
    CUptiResult (*FlushAll)(uint32_t) = nullptr;
    CUptiResult (*GetNextRecord)(uint8_t*, size_t, CUpti_Activity**) = nullptr;
    CUptiResult (*GetNumDroppedRecords)(CUcontext, uint32_t, size_t*) = nullptr;
    CUptiResult (*GetResultString)(CUptiResult, const char**) = nullptr;
} C;

int fail(const std::string& m) {
    g_err = m;
    return -1;
}

int cupti_fail(const char* what, CUptiResult r) {
    const char* s = nullptr;
    if (C.GetResultString) C.GetResultString(r, &s);
    return fail(std::string(what) + ": " + (s ? s : "CUPTI error") + " (" + std::to_string((int)r) + ")");
}

int load_cupti() {
    if (C.h) return 0;
    const char* names[] = {"libcupti.so.12", "libcupti.so", "/usr/local/cuda/targets/x86_64-linux/lib/libcupti.so.12",
                           "/usr/local/cuda-12.9/targets/x86_64-linux/lib/libcupti.so.12", "/usr/local/cuda/extras/CUPTI/lib64/libcupti.so.12"};
    void* h = nullptr;
    for (const char* n : names)
        if ((h = dlopen(n, RTLD_NOW | RTLD_GLOBAL))) break;
    if (!h) return fail(std::string("cannot load libcupti: ") + dlerror());
#define SYM(field, name)                                             \
    *(void**)(&C.field) = dlsym(h, name);                            \
    if (!C.field) return fail(std::string("libcupti lacks ") + name)
    SYM(RegisterCallbacks, "cuptiActivityRegisterCallbacks");
    SYM(Enable, "cuptiActivityEnable");
    SYM(Disable, "cuptiActivityDisable");
    SYM(FlushAll, "cuptiActivityFlushAll");
    SYM(GetNextRecord, "cuptiActivityGetNextRecord");
    SYM(GetNumDroppedRecords, "cuptiActivityGetNumDroppedRecords");
    SYM(GetResultString, "cuptiGetResultString");
#undef SYM
    C.h = h;
    return 0;
}

constexpr size_t kBufBytes = 8u << 20;

// kernel names seen, for the optional raw dump (SET_TRACE_DUMP=<file>: one CSV line per record)
std::vector<std::string> g_names{""};
uint32_t name_id(const char* n) {
    if (!n) return 0;
    for (size_t i = 1; i < g_names.size(); ++i)
        if (g_names[i] == n) return (uint32_t)i;
    g_names.emplace_back(n);
    return (uint32_t)g_names.size() - 1;
}

void CUPTIAPI buffer_requested(uint8_t** buffer, size_t* size, size_t* max_records) {
    void* p = nullptr;
    if (posix_memalign(&p, 8, kBufBytes) != 0) p = nullptr;
    *buffer = (uint8_t*)p;
    *size = p ? kBufBytes : 0;
    *max_records = 0;
}

void CUPTIAPI buffer_completed(CUcontext ctx, uint32_t stream_id, uint8_t* buffer, size_t, size_t valid) {
    if (buffer && valid > 0) {
        std::lock_guard<std::mutex> lk(g_mu);
        CUpti_Activity* rec = nullptr;
        while (C.GetNextRecord(buffer, valid, &rec) == CUPTI_SUCCESS) {
            set_trace_rec r{};
            switch (rec->kind) {
                case CUPTI_ACTIVITY_KIND_KERNEL:
                case CUPTI_ACTIVITY_KIND_CONCURRENT_KERNEL: {
                    auto* k = (CUpti_ActivityKernel9*)rec;
                    r.stream = k->streamId;
                    r.job = k->correlationId;
                    r.kind = (k->name && strstr(k->name, "set_k_signal")) ? 1u : 0u;
                    r.reserved = name_id(k->name);
                    r.start_ns = k->start;
                    r.end_ns = k->end;
                    break;
                }
                case CUPTI_ACTIVITY_KIND_MEMCPY: {
                    auto* m = (CUpti_ActivityMemcpy6*)rec;
                    r.stream = m->streamId;
                    r.job = m->correlationId;
                    r.kind = 2;
                    r.start_ns = m->start;
                    r.end_ns = m->end;
                    break;
                }
                case CUPTI_ACTIVITY_KIND_MEMSET: {
                    auto* m = (CUpti_ActivityMemset4*)rec;
                    r.stream = m->streamId;
                    r.job = m->correlationId;
                    r.kind = 3;
                    r.start_ns = m->start;
                    r.end_ns = m->end;
                    break;
                }
                default:
                    continue;
            }
            if (r.end_ns >= r.start_ns && r.start_ns != 0) g_recs.push_back(r);
        }
        size_t dropped = 0;
        if (C.GetNumDroppedRecords(ctx, stream_id, &dropped) == CUPTI_SUCCESS) g_dropped += dropped;
    }
    free(buffer);
}

set_gap_summary summarise(std::vector<double>& g) {
    set_gap_summary s{};
    s.count = g.size();
    if (g.empty()) return s;
    std::sort(g.begin(), g.end());
    double sum = 0;
    for (double v : g) sum += v;
    s.mean_us = sum / (double)g.size();
    auto q = [&](double p) { return g[std::min(g.size() - 1, (size_t)(p * (double)(g.size() - 1) + 0.5))]; };
    s.p50_us = q(0.50);
    s.p99_us = q(0.99);
    s.max_us = g.back();
    return s;
}

}  // namespace

extern "C" const char* set_trace_error(void) { return g_err.c_str(); }

extern "C" int set_trace_reduce(const set_trace_rec* recs, uint64_t n, set_trace_stats* out) {
    if (!out || (n > 0 && !recs)) return fail("set_trace_reduce: NULL argument");
    memset(out, 0, sizeof(*out));
    if (n == 0) return 0;
    std::vector<set_trace_rec> v(recs, recs + n);
    std::vector<double> kk, intra, inter, any;
    uint64_t t_first = UINT64_MAX, t_last = 0;
    double ksum = 0, opsum = 0;
    uint64_t nk = 0;
    for (auto& r : v) {
        t_first = std::min(t_first, r.start_ns);
        t_last = std::max(t_last, r.end_ns);
        opsum += (double)(r.end_ns - r.start_ns) * 1e-3;
        switch (r.kind) {
            case 0: out->kernels++; ksum += (double)(r.end_ns - r.start_ns) * 1e-3; nk++; break;
            case 1: out->kernels++; out->signal_kernels++; break;
            case 2: out->memcpys++; break;
            default: out->memsets++; break;
        }
    }
    // ---- every consecutive pair on one CUPTI stream id (the raw view; negative = overlap = 0)
    std::sort(v.begin(), v.end(), [](const set_trace_rec& a, const set_trace_rec& b) {
        if (a.stream != b.stream) return a.stream < b.stream;
        if (a.start_ns != b.start_ns) return a.start_ns < b.start_ns;
        return a.end_ns < b.end_ns;
    });
    for (size_t i = 1; i < v.size(); ++i)
        if (v[i - 1].stream == v[i].stream)
            any.push_back(v[i].start_ns > v[i - 1].end_ns ? (double)(v[i].start_ns - v[i - 1].end_ns) * 1e-3 : 0.0);
    // ---- jobs: the records of one graph launch share its correlation id.  CUPTI gives the parallel branches of a job graph
    // (memset || H2D, two D2H leaves) stream ids of their own, so a job's WORK STREAM is the id most of its kernels ran under,
    // and everything below is per job, not per CUPTI stream id.
    std::sort(v.begin(), v.end(), [](const set_trace_rec& a, const set_trace_rec& b) {
        if (a.job != b.job) return a.job < b.job;
        if (a.start_ns != b.start_ns) return a.start_ns < b.start_ns;
        return a.end_ns < b.end_ns;
    });
    struct Job {
        uint32_t stream;
        uint64_t start, end;
    };
    std::vector<Job> jobs;
    for (size_t a = 0; a < v.size();) {
        size_t b = a;
        while (b < v.size() && v[b].job == v[a].job) ++b;
        Job jb{v[a].stream, v[a].start_ns, v[a].end_ns};
        std::map<uint32_t, int> votes;
        uint64_t reach = v[a].end_ns;      // latest end among the job's ops so far
        const set_trace_rec* last_kernel = nullptr;
        for (size_t i = a; i < b; ++i) {
            const set_trace_rec& r = v[i];
            jb.end = std::max(jb.end, r.end_ns);
            if (r.kind <= 1) votes[r.stream]++;
            if (i > a) intra.push_back(r.start_ns > reach ? (double)(r.start_ns - reach) * 1e-3 : 0.0);
            reach = std::max(reach, r.end_ns);
            if (r.kind == 0) {
                // stage kernel -> next stage kernel of the same job, SIGNED: a programmatic (PDL) edge lets the next kernel
                // start before its predecessor has ended, which shows as a negative gap instead of a flat zero
                if (last_kernel) {
                    double g = ((double)r.start_ns - (double)last_kernel->end_ns) * 1e-3;
                    kk.push_back(g);
                    if (g < 0) out->kernel_kernel_overlapped++;
                }
                last_kernel = &r;
            } else if (r.kind != 1) {
                last_kernel = nullptr;  // a copy or memset in between: not a kernel-to-kernel hand-off
            }
        }
        int best = 0;
        for (auto& kv : votes)
            if (kv.second > best) {
                best = kv.second;
                jb.stream = kv.first;
            }
        jobs.push_back(jb);
        a = b;
    }
    out->jobs = jobs.size();
    std::sort(jobs.begin(), jobs.end(), [](const Job& a, const Job& b) { return a.stream != b.stream ? a.stream < b.stream : a.start < b.start; });
    for (size_t i = 0; i < jobs.size(); ++i) {
        if (i == 0 || jobs[i - 1].stream != jobs[i].stream) {
            out->streams++;
            continue;
        }
        inter.push_back(jobs[i].start > jobs[i - 1].end ? (double)(jobs[i].start - jobs[i - 1].end) * 1e-3 : 0.0);
    }
    // union of all activity intervals, over all streams
    std::vector<std::pair<uint64_t, uint64_t>> iv;
    iv.reserve(v.size());
    for (auto& r : v) iv.emplace_back(r.start_ns, r.end_ns);
    std::sort(iv.begin(), iv.end());
    uint64_t busy = 0, cs = iv[0].first, ce = iv[0].second;
    for (size_t i = 1; i < iv.size(); ++i) {
        if (iv[i].first <= ce) {
            ce = std::max(ce, iv[i].second);
        } else {
            busy += ce - cs;
            cs = iv[i].first;
            ce = iv[i].second;
        }
    }
    busy += ce - cs;
    out->wall_us = (double)(t_last - t_first) * 1e-3;
    out->busy_us = (double)busy * 1e-3;
    out->idle_frac = out->wall_us > 0 ? 1.0 - out->busy_us / out->wall_us : 0.0;
    out->kernel_mean_us = nk ? ksum / (double)nk : 0.0;
    out->sum_op_us = opsum;
    out->kernel_kernel = summarise(kk);
    out->intra_job = summarise(intra);
    out->inter_job = summarise(inter);
    out->any_op = summarise(any);
    return 0;
}

extern "C" int set_trace_start(void) {
    if (g_on) return fail("set_trace_start: already tracing");
    if (int rc = load_cupti()) return rc;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        g_recs.clear();
        g_dropped = 0;
    }
    static bool registered = false;
    if (!registered) {
        CUptiResult r = C.RegisterCallbacks(buffer_requested, buffer_completed);
        if (r != CUPTI_SUCCESS) return cupti_fail("cuptiActivityRegisterCallbacks", r);
        registered = true;
    }
    const CUpti_ActivityKind kinds[] = {CUPTI_ACTIVITY_KIND_CONCURRENT_KERNEL, CUPTI_ACTIVITY_KIND_MEMCPY, CUPTI_ACTIVITY_KIND_MEMSET};
    for (auto k : kinds) {
        CUptiResult r = C.Enable(k);
        if (r != CUPTI_SUCCESS) return cupti_fail("cuptiActivityEnable", r);
    }
    g_on = true;
    return 0;
}

extern "C" int set_trace_stop(set_trace_stats* out) {
    if (!g_on) return fail("set_trace_stop: not tracing");
    g_on = false;
    CUptiResult r = C.FlushAll(1 /* CUPTI_ACTIVITY_FLAG_FLUSH_FORCED */);
    const CUpti_ActivityKind kinds[] = {CUPTI_ACTIVITY_KIND_CONCURRENT_KERNEL, CUPTI_ACTIVITY_KIND_MEMCPY, CUPTI_ACTIVITY_KIND_MEMSET};
    for (auto k : kinds) C.Disable(k);
    if (r != CUPTI_SUCCESS) return cupti_fail("cuptiActivityFlushAll", r);
    std::vector<set_trace_rec> recs;
    uint64_t dropped;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        recs.swap(g_recs);
        dropped = g_dropped;
    }
    if (const char* path = getenv("SET_TRACE_DUMP")) {
        if (FILE* f = fopen(path, "a")) {
            fprintf(f, "# stream,job,kind,start_ns,end_ns,name\n");
            for (auto& r : recs)
                fprintf(f, "%u,%u,%u,%llu,%llu,%s\n", r.stream, r.job, r.kind, (unsigned long long)r.start_ns, (unsigned long long)r.end_ns,
                        r.reserved < g_names.size() ? g_names[r.reserved].c_str() : "");
            fclose(f);
        }
    }
    int rc = set_trace_reduce(recs.data(), recs.size(), out);
    if (rc == 0 && out) out->dropped = dropped;
    return rc;
}
