// set_selftest.cpp -- host-only self tests of the lock-free structures and of Algorithms 1-3 against a
// SIMULATED device (threads stand in for the CUDA driver's callback thread).  No CUDA call is made, so these
// run in the CPU-only test tier.  Declared in include/set.h ("Host-only self tests").
#include <atomic>
#include <chrono>
#include <mutex>
#include <thread>
#include <vector>

#include "../../include/set.h"
#include "set_core.hpp"

using namespace setrt;

extern "C" int set_selftest_find_order(int b, int w, uint64_t nonempty) {
    if (b < 1 || b > 64 || w < 0 || w >= b) return -2;
    return Scheduler::find_order(b, w, nonempty);
}

extern "C" int64_t set_selftest_ring(int capacity, int producers, int consumers, int64_t items_per_producer) {
    if (capacity < 1 || producers < 1 || consumers < 1 || items_per_producer < 0) return -1;
    Ring<uint64_t> ring((size_t)capacity);
    const int64_t total = (int64_t)producers * items_per_producer;
    std::vector<std::atomic<uint8_t>> seen((size_t)total);
    for (auto& s : seen) s.store(0);
    std::atomic<int64_t> popped{0}, errors{0};
    std::vector<std::thread> th;
    for (int p = 0; p < producers; ++p)
        th.emplace_back([&, p] {
            for (int64_t i = 0; i < items_per_producer; ++i) {
                uint64_t tok = (uint64_t)p * (uint64_t)items_per_producer + (uint64_t)i;
                Backoff bo;
                while (!ring.try_push(tok)) bo.pause();
            }
        });
    for (int c = 0; c < consumers; ++c)
        th.emplace_back([&] {
            uint64_t last_from[64];
            for (auto& l : last_from) l = 0;
            Backoff bo;
            while (popped.load(std::memory_order_relaxed) < total) {
                uint64_t tok;
                if (!ring.try_pop(tok)) {
                    bo.pause();
                    continue;
                }
                bo = Backoff();
                if (tok >= (uint64_t)total) { errors.fetch_add(1); continue; }
                if (seen[(size_t)tok].fetch_add(1) != 0) errors.fetch_add(1);  // delivered twice
                // FIFO per producer as observed by ONE consumer: tokens of a producer arrive in order
                int p = (int)(tok / (uint64_t)(items_per_producer ? items_per_producer : 1));
                if (p < 64) {
                    if (last_from[p] > tok + 1 && last_from[p] != 0) errors.fetch_add(1);
                    last_from[p] = tok + 1;
                }
                popped.fetch_add(1, std::memory_order_relaxed);
            }
        });
    for (auto& t : th) t.join();
    for (auto& s : seen)
        if (s.load() != 1) errors.fetch_add(1);
    uint64_t dummy;
    if (ring.try_pop(dummy)) errors.fetch_add(1);  // must be empty now
    return -errors.load();
}

namespace {

// Simulated device: launch() hands (slot, due time) to completer threads, which call on_complete(slot).
class SimBackend : public Backend {
  public:
    SimBackend(int slots, int epp, int completers, int64_t jobs, uint32_t seed, bool polled)
        : b_(slots), epp_(epp), jobs_(jobs), seed_(seed), inbox_((size_t)slots + 1), polled_(polled) {
        flags_.assign((size_t)slots * kFlagStride, 0u);
        bound_slot_.assign((size_t)slots * epp, -1);
        for (int e = 0; e < slots * epp; ++e) bound_slot_[(size_t)e] = e / epp;  // execs start tied to M_home
        exec_busy_ = std::vector<std::atomic<int>>((size_t)slots * epp);
        slot_busy_ = std::vector<std::atomic<int>>((size_t)slots);
        done_count_ = std::vector<std::atomic<int>>((size_t)jobs);
        for (auto& a : exec_busy_) a.store(0);
        for (auto& a : slot_busy_) a.store(0);
        for (auto& a : done_count_) a.store(0);
        ncompleters_ = completers;
    }
    void attach(Scheduler* s) {
        sched_ = s;
        for (int c = 0; c < ncompleters_; ++c) threads_.emplace_back([this] { completer(); });
    }
    void shutdown() {
        stop_.store(true);
        for (auto& t : threads_) t.join();
        threads_.clear();
    }
    int bind(int exec, int slot, JobDesc& job, bool* pinned) override {
        *pinned = false;
        if (exec_busy_[(size_t)exec].load() != 0) errors.fetch_add(1);  // never update an exec that is in flight
        bound_slot_[(size_t)exec] = slot;
        (void)job;
        binds.fetch_add(1);
        return 0;
    }
    int launch(int exec, int slot, const JobDesc& job) override {
        if (bound_slot_[(size_t)exec] != slot) errors.fetch_add(1);  // G must be bound to the launching slot's M_w
        if (slot >= in_service.load() || exec / epp_ >= in_service.load()) errors.fetch_add(1);  // a retired slot or one of its execs
        if (slot_busy_[(size_t)slot].exchange(1) != 0) errors.fetch_add(1);  // one job per slot at a time
        if (exec_busy_[(size_t)exec].exchange(1) != 0) errors.fetch_add(1);
        int64_t inflight = inflight_.fetch_add(1) + 1;
        if (inflight > b_) errors.fetch_add(1);  // bounded in-flight executables
        // pseudo-random service time 0..~40 us keyed by the job id: completions come out of order
        uint32_t h = (uint32_t)job.id * 2654435761u ^ seed_;
        h ^= h >> 15;
        uint64_t due = now_ns() + (uint64_t)(h % 40u) * 1000ull;
        Item it{slot, exec, job.id, due};
        inbox_.push(it);
        return 0;
    }
    void finish(int exec, int slot, const JobDesc& job) override {
        if (job.id < (uint64_t)jobs_) done_count_[(size_t)job.id].fetch_add(1);
        exec_busy_[(size_t)exec].store(0);
        slot_busy_[(size_t)slot].store(0);
        inflight_.fetch_sub(1);
    }
    // polled completion: the completer threads play the GPU and store the slot's word
    volatile uint32_t* done_flags() override { return polled_ ? flags_.data() : nullptr; }
    int64_t check_all_done_once() {
        int64_t bad = 0;
        for (auto& d : done_count_)
            if (d.load() != 1) ++bad;
        return bad;
    }
    std::atomic<int64_t> errors{0}, binds{0};
    std::atomic<int> in_service{1 << 30};  // Scheduler::retire_slots: slots below this number may run jobs

  private:
    struct Item {
        int slot, exec;
        uint64_t id, due;
    };
    void completer() {
        std::vector<Item> held;
        Backoff bo;
        while (!stop_.load(std::memory_order_acquire) || !held.empty() || !inbox_.empty_approx()) {
            Item it;
            while (inbox_.try_pop(it)) held.push_back(it);
            uint64_t t = now_ns();
            bool any = false;
            for (size_t i = 0; i < held.size();) {
                if (held[i].due <= t) {
                    int slot = held[i].slot;
                    held[i] = held.back();
                    held.pop_back();
                    if (polled_)
                        __atomic_store_n(&flags_[(size_t)slot * kFlagStride], 1u, __ATOMIC_RELEASE);
                    else
                        sched_->on_complete(slot);
                    any = true;
                } else {
                    ++i;
                }
            }
            if (any)
                bo = Backoff();
            else
                bo.pause();
        }
    }
    int b_, epp_;
    int64_t jobs_;
    uint32_t seed_;
    int ncompleters_ = 1;
    Ring<Item> inbox_;
    bool polled_ = false;
    std::vector<uint32_t> flags_;
    std::vector<int> bound_slot_;
    std::vector<std::atomic<int>> exec_busy_, slot_busy_, done_count_;
    std::atomic<int64_t> inflight_{0};
    std::atomic<bool> stop_{false};
    Scheduler* sched_ = nullptr;
    std::vector<std::thread> threads_;
};

}  // namespace

extern "C" int64_t set_selftest_scheduler(int num_streams, int max_inflight, int queue_capacity, int num_dispatchers,
                                          int submitters, int64_t jobs, uint32_t seed, uint64_t* out_steals) {
    if (num_streams < 1 || max_inflight < 1 || queue_capacity < 1 || num_dispatchers < 1 || submitters < 1 || jobs < 0)
        return -1;
    int b = ((max_inflight + num_streams - 1) / num_streams) * num_streams;
    int policy = (seed & 1) ? Scheduler::kRetarget : Scheduler::kSwap;
    SimBackend be(b, queue_capacity + 1, 2, jobs, seed, /*polled=*/(seed & 2) != 0);
    int64_t rc = 0;
    {
        Scheduler sched(&be, num_streams, b, queue_capacity, num_dispatchers, policy, 20, /*poller=*/(seed >> 2) & 1);
        sched.set_bind_at_launch((seed >> 3) & 1);
        const int keep = ((seed >> 4) & 1) ? num_streams : b;  // seed bit 4: a loop pipeline's geometry (slot-bound, one slot per stream)
        if (keep < b) {
            sched.set_slot_bound(true);
            sched.retire_slots(keep);
            be.in_service.store(keep);
        }
        be.attach(&sched);
        std::atomic<int64_t> next{0};
        std::vector<std::thread> subs;
        std::atomic<int64_t> submit_errors{0}, would_block{0};
        for (int s = 0; s < submitters; ++s)
            subs.emplace_back([&] {
                for (;;) {
                    int64_t j = next.fetch_add(1);
                    if (j >= jobs) break;
                    JobDesc d;
                    d.id = (uint64_t)j;
                    if ((seed >> 5) & 1) {  // seed bit 5: non-blocking submits, retried while every executable is taken (set_try_submit_dims)
                        int rc;
                        while ((rc = sched.submit(d, /*blocking=*/false)) == Scheduler::kWouldBlock) {
                            would_block.fetch_add(1);
                            std::this_thread::yield();
                        }
                        if (rc != 0) submit_errors.fetch_add(1);
                    } else if (sched.submit(d) != 0) {
                        submit_errors.fetch_add(1);
                    }
                }
            });
        for (auto& t : subs) t.join();
        int drc = sched.drain();
        if (drc != 0) rc = -100 + drc;
        if (submit_errors.load() != 0) rc = -2;
        CoreStats& st = sched.stats();
        if ((int64_t)st.completed.load() != jobs || (int64_t)st.submitted.load() != jobs) rc = -3;
        if ((int64_t)st.max_inflight.load() > keep) rc = -4;
        if (out_steals) *out_steals = st.steals.load();
        sched.stop();
        be.shutdown();
    }
    if (be.errors.load() != 0) rc = -5;
    if (be.check_all_done_once() != 0) rc = -6;
    return rc;
}
