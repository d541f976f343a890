// set_core.hpp -- the SET scheduler proper: Algorithms 1-3 of arxiv/paper_2606_05495
// over an abstract device backend.  Host-side integer/pointer work only; every CUDA call lives in the
// backend (set_cuda.cpp).  The same core runs against a simulated device in set_selftest.cpp so that the
// lock-free logic is testable without a GPU.
//
// Vocabulary:
//   slot w      worker W_w = (stream S_{w mod S}, device buffers M_w, execs bound to M_w)
//   Q_w         per-slot queue of PREPARED jobs (exec already updated for the job)   -- Ring<Prepared>
//   W_pool      free worker pool: ids of slots with nothing in flight               -- Ring<int>
//   c_next      next-job counter (Alg. 1), c_done finished-job counter (Alg. 3)
#pragma once
#include <atomic>
#include <cerrno>
#include <climits>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <memory>
#include <thread>
#include <vector>

#include <linux/futex.h>
#include <sys/syscall.h>
#include <time.h>
#include <unistd.h>

#include "set_ring.hpp"

namespace setrt {

inline uint64_t now_ns() {
    timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (uint64_t)ts.tv_sec * 1000000000ull + (uint64_t)ts.tv_nsec;
}

inline void cpu_relax() {
#if defined(__x86_64__) || defined(__i386__)
    __builtin_ia32_pause();
#else
    asm volatile("" ::: "memory");
#endif
}

// Event count: sleepers block in the kernel (futex) only after spinning for spin_ns.
// notify() costs one atomic increment and, only if somebody sleeps, one syscall -- this is the
// notify_one() of Algorithm 3 l.3.
class EventCount {
  public:
    uint32_t prepare() const { return epoch_.load(std::memory_order_acquire); }
    // Wait until the epoch differs from `seen` (or, with timeout_ns != 0, until about that much time has passed
    // in the kernel).  Returns true if the thread went to sleep.  Callers re-check their condition in a loop.
    bool wait(uint32_t seen, uint64_t spin_ns, uint64_t timeout_ns = 0) {
        uint64_t t0 = now_ns();
        for (int i = 0;; ++i) {
            if (epoch_.load(std::memory_order_acquire) != seen) return false;
            cpu_relax();
            if ((i & 63) == 63 && now_ns() - t0 >= spin_ns) break;
        }
        sleepers_.fetch_add(1, std::memory_order_seq_cst);
        bool slept = false;
        timespec ts{(time_t)(timeout_ns / 1000000000ull), (long)(timeout_ns % 1000000000ull)};
        while (epoch_.load(std::memory_order_seq_cst) == seen) {
            slept = true;
            long rc = syscall(SYS_futex, reinterpret_cast<uint32_t*>(&epoch_), FUTEX_WAIT_PRIVATE, seen,
                              timeout_ns ? &ts : nullptr, nullptr, 0);
            if (timeout_ns && rc == -1 && errno == ETIMEDOUT) break;
        }
        sleepers_.fetch_sub(1, std::memory_order_seq_cst);
        return slept;
    }
    void notify_all() {
        epoch_.fetch_add(1, std::memory_order_seq_cst);
        if (sleepers_.load(std::memory_order_seq_cst) > 0)
            syscall(SYS_futex, reinterpret_cast<uint32_t*>(&epoch_), FUTEX_WAKE_PRIVATE, INT_MAX, nullptr, nullptr, 0);
    }

  private:
    alignas(kCacheLine) std::atomic<uint32_t> epoch_{0};
    alignas(kCacheLine) std::atomic<uint32_t> sleepers_{0};
};
static_assert(sizeof(std::atomic<uint32_t>) == 4, "futex word");

struct JobDesc {
    uint64_t id = 0;
    const void* in = nullptr;
    void* out = nullptr;
    uint32_t dims[4] = {1, 1, 1, 1};
};

// Queue entry: a fully prepared graph executable, not a task index.
struct Prepared {
    int32_t exec = -1;  // global exec index; its free list is that of slot exec / execs_per_slot
    int32_t home = -1;  // slot whose memory M_home the exec is bound to
    JobDesc job;
};

// Device side of the scheduler.  bind = UpdateGraphParams (Alg. 1 l.4, Alg. 2 l.20); launch = GraphLaunch +
// AddCallback (Alg. 2 l.21-22).  launch() must arrange for Scheduler::on_complete(slot) to be called exactly
// once, from any thread, when the job's last operation has finished.
class Backend {
  public:
    virtual ~Backend() = default;
    // Returns 0 or a negative set_status.  `pinned_to_exec`: true if the job's data now lives in storage tied
    // to this exec (pageable staging), so a thief must retarget this very exec instead of swapping.
    virtual int bind(int exec, int slot, JobDesc& job, bool* pinned_to_exec) = 0;
    virtual int launch(int exec, int slot, const JobDesc& job) = 0;
    // Bind-at-launch mode only: the checks of bind() that concern the job alone (per-job sizes), made at submit time so
    // that the caller still gets SET_ERR_SIZE synchronously.  Returns 0 or a negative set_status.
    virtual int validate(const JobDesc&) { return 0; }
    // Called on the completing thread before the slot is released (e.g. staged D2H -> caller memory).
    virtual void finish(int exec, int slot, const JobDesc& job) = 0;
    // Called from a blocked submit/drain every kPollNs: report an asynchronous device failure (a faulting stage
    // kernel) as a negative set_status.  The driver never runs a host function behind failed work, so without
    // this check a fault would leave c_done short of c_submitted forever.
    virtual int poll() { return 0; }
    // Flag-polled completion (SET_CB_FLAG_POLL): non-null => the last node of every job graph stores a non-zero
    // word to done_flags()[slot * kFlagStride] (pinned host memory the GPU writes directly); no host function is
    // enqueued, the dispatcher itself watches the words and runs Algorithm 3.  The core clears the word before launch().
    virtual volatile uint32_t* done_flags() { return nullptr; }
};

constexpr int kFlagStride = 16;  // one 64-byte line per slot: the GPU's write invalidates only that slot's line

struct CoreStats {
    std::atomic<uint64_t> submitted{0}, completed{0}, launched{0}, steals{0}, submit_stalls{0},
        dispatcher_sleeps{0}, ns_submit{0}, ns_launch{0}, ns_callback{0}, max_inflight{0};
};

class Scheduler {
  public:
    enum StealPolicy { kSwap = 0, kRetarget = 1 };

    // poller: with flag-polled completion, 1 = a thread of its own watches the completion words and runs Algorithm 3, so that
    // the dispatcher threads do nothing but FindJob + LaunchJob (the dispatcher was the bottleneck of the short-job configs:
    // 1.9 us of cudaGraphLaunch + 1 us of polling and completion per job); 0 = the dispatchers poll between launches.
    Scheduler(Backend* be, int num_streams, int slots, int queue_capacity, int num_dispatchers, int steal_policy,
              int spin_us, int poller = 0)
        : be_(be),
          S_(num_streams),
          b_(slots),
          q_(queue_capacity),
          epp_(queue_capacity + 1),
          steal_policy_(steal_policy),
          spin_ns_((uint64_t)spin_us * 1000ull) {
        queues_.reset(new PaddedRing<Prepared>[b_]);
        free_execs_.reset(new PaddedRing<int>[b_]);
        running_.reset(new Running[b_]);
        flags_ = be_->done_flags();
        for (int w = 0; w < b_; ++w) {
            queues_[w].r.init((size_t)epp_ + 1);
            free_execs_[w].r.init((size_t)epp_ * 2);  // room for migrated execs under kRetarget
            for (int k = 0; k < epp_; ++k) free_execs_[w].r.push(w * epp_ + k);
        }
        launched_.reset(new StreamOrder[S_]);
        for (int s = 0; s < S_; ++s) launched_[s].q.init((size_t)b_ + 1);
        pool_.init((size_t)b_ + 1);
        // the main thread initialises all workers; all of them start idle.
        for (int w = 0; w < b_; ++w) pool_.push(w);
        n_free_.store(b_, std::memory_order_relaxed);
        active_ = b_;
        own_poller_ = flags_ != nullptr && poller != 0;
        for (int d = 0; d < num_dispatchers; ++d) dispatchers_.emplace_back([this] { dispatcher_loop(); });
        if (own_poller_) dispatchers_.emplace_back([this] { poller_loop(); });
    }

    ~Scheduler() { stop(); }

    void stop() {
        bool expected = false;
        if (!stop_.compare_exchange_strong(expected, true)) return;
        work_ec_.notify_all();
        poll_ec_.notify_all();
        for (auto& t : dispatchers_) t.join();
        dispatchers_.clear();
    }

    // Executables that cannot leave their slot (a job graph with a conditional loop is built per slot): a thief may only
    // use an executable of its OWN slot; if it has none free at this instant it hands the job back to the victim's queue.
    void set_slot_bound(bool v) { slot_bound_.store(v, std::memory_order_release); }
    // Bind at launch: submit() only reserves an executable of the slot and queues the job's description; UpdateGraphParams runs
    // on the dispatcher thread right before GraphLaunch -- the "JIT update" of PAPER.md:122 applied to every job.  All driver
    // calls of a job then come from ONE thread: graph updates and launches go through the same driver lock, and issued from two
    // threads they cost 0.6 + 2.3 us per job on B200, from one thread 0.3 + 1.7 us.
    void set_bind_at_launch(bool v) { lazy_bind_.store(v, std::memory_order_release); }

    // Take slots keep .. b-1 out of service.  Only before the first job is submitted (nothing queued, nothing in flight): their
    // executables leave the free lists, so Algorithm 1 never queues a job on them, and they leave W_pool, so they never
    // dispatch or steal.  The backend asks for this where more slots than CUDA streams cost throughput.
    void retire_slots(int keep) {
        if (keep < 1 || keep >= b_) return;
        std::vector<int> ws;
        int w = -1, e = -1;
        while (pool_.try_pop(w)) ws.push_back(w);
        int kept = 0;
        for (int x : ws)
            if (x < keep) {
                pool_.push(x);
                ++kept;
            }
        n_free_.store(kept, std::memory_order_seq_cst);
        for (w = keep; w < b_; ++w)
            while (free_execs_[w].r.try_pop(e)) {
            }
        active_ = keep;
    }
    int active_slots() const { return active_; }

    int slots() const { return b_; }
    int execs_per_slot() const { return epp_; }
    CoreStats& stats() { return stats_; }
    int error() const { return err_.load(std::memory_order_acquire); }
    void set_error(int e) {
        int zero = 0;
        err_.compare_exchange_strong(zero, e);
        done_ec_.notify_all();
        space_ec_.notify_all();
    }

    // ---- Algorithm 1: job submitter --------------------------------------
    // The paper's submitter claims job indices from a shared array with compare_exchange(c_next, id, id+1);
    // here the caller hands the job over, so the claim degenerates to a fetch_add that yields the ticket used
    // to pick the first queue to look at ("monitors all queues for available slots").
    static constexpr int kWouldBlock = -6;  // SET_ERR_BUSY: a non-blocking submit found no free executable
    int submit(JobDesc job, bool blocking = true) {
        uint64_t t0 = now_ns();
        if (int e = error()) return e;
        uint64_t ticket = c_next_.fetch_add(1, std::memory_order_relaxed);
        int start = (int)(ticket % (uint64_t)b_);
        int exec = -1, slot = -1;
        for (;;) {
            uint32_t seen = space_ec_.prepare();
            for (int k = 0; k < b_; ++k) {  // "Q_i not full" == slot i still has an unused exec
                int i = start + k;
                if (i >= b_) i -= b_;
                if (free_execs_[i].r.try_pop(exec)) {
                    slot = i;
                    break;
                }
            }
            if (slot >= 0) break;
            if (int e = error()) return e;
            if (!blocking) return kWouldBlock;  // nothing was taken, nothing to undo (the ticket only picks where the scan starts)
            stats_.submit_stalls.fetch_add(1, std::memory_order_relaxed);
            if (space_ec_.wait(seen, spin_ns_, kPollNs))
                if (int e = be_->poll()) set_error(e);
        }
        Prepared p;
        p.exec = exec;
        p.home = slot;
        p.job = job;
        bool pinned = false;
        const bool lazy = lazy_bind_.load(std::memory_order_acquire);
        int rc = lazy ? be_->validate(p.job) : be_->bind(exec, slot, p.job, &pinned);  // UpdateGraphParams(J_id, i)
        if (lazy) p.home |= kUnboundBit;
        if (rc != 0) {
            free_execs_[slot].r.push(exec);
            space_ec_.notify_all();
            if (rc != -5 /*SET_ERR_SIZE is per job, not sticky*/) set_error(rc);
            return rc;
        }
        if (pinned) p.home |= kPinnedBit;
        stats_.submitted.fetch_add(1, std::memory_order_relaxed);
        c_submitted_.fetch_add(1, std::memory_order_release);
        queues_[slot].r.push(p);  // room is guaranteed: entries are bounded by the slot's exec count
        n_queued_.fetch_add(1, std::memory_order_seq_cst);
        work_ec_.notify_all();
        stats_.ns_submit.fetch_add(now_ns() - t0, std::memory_order_relaxed);
        return 0;
    }

    // ---- Algorithm 3: asynchronous resource return ------------------------
    // Runs on the CUDA driver's callback thread (or a simulated completer).  No CUDA call in here.
    void on_complete(int w) {
        uint64_t t0 = now_ns();
        Running& r = running_[w];
        be_->finish(r.exec, w, r.job);
        int exec = r.exec;
        r.exec = -1;
        r.state.store(0, std::memory_order_release);
        inflight_.fetch_sub(1, std::memory_order_seq_cst);
        free_execs_[exec / epp_].r.push(exec);  // the exec returns to its home free list
        space_ec_.notify_all();
        pool_.push(w);  // W_pool.push(w_id)
        n_free_.fetch_add(1, std::memory_order_seq_cst);
        work_ec_.notify_all();  // notify_one()
        stats_.completed.fetch_add(1, std::memory_order_relaxed);
        uint64_t done = c_done_.fetch_add(1, std::memory_order_acq_rel) + 1;  // c_done.fetch_add(1)
        if (done == c_submitted_.load(std::memory_order_acquire)) done_ec_.notify_all();
        stats_.ns_callback.fetch_add(now_ns() - t0, std::memory_order_relaxed);
    }

    // ---- A8 drain: wait for c_done == c_submitted ----------------------------------------------------------
    int drain() {
        uint64_t err_t0 = 0;
        for (;;) {
            uint32_t seen = done_ec_.prepare();
            if (c_done_.load(std::memory_order_acquire) == c_submitted_.load(std::memory_order_acquire)) break;
            if (error()) {
                // A failed context may never deliver its callbacks: give in-flight work a bounded grace
                // period, then return the error instead of hanging (set.h "set_drain still returns").
                if (n_queued_.load() <= 0 && inflight_.load() <= 0) break;
                if (err_t0 == 0) err_t0 = now_ns();
                if (now_ns() - err_t0 > 2000000000ull) break;
                timespec ts{0, 200000};
                nanosleep(&ts, nullptr);
                continue;
            }
            if (done_ec_.wait(seen, spin_ns_, kPollNs))
                if (int e = be_->poll()) set_error(e);
        }
        return error();
    }

    // FindJob's victim order, exposed for the host-only self test (Alg. 2 l.8-17).
    static int find_order(int b, int w, uint64_t nonempty) {
        if (nonempty >> w & 1) return w;
        for (int k = 1; k < b; ++k) {
            int v = (w + k) % b;
            if (nonempty >> v & 1) return v;
        }
        return -1;
    }

  private:
    static constexpr int32_t kPinnedBit = 1 << 30;
    static constexpr int32_t kUnboundBit = 1 << 29;
    static constexpr uint64_t kPollNs = 20000000ull;  // 20 ms
    template <typename T>
    struct alignas(kCacheLine) PaddedRing {
        Ring<T> r;
    };
    // Slots in the order their jobs were launched on one stream.  A stream completes its graphs in launch order, so a
    // polling dispatcher only has to watch the OLDEST in-flight slot of each stream: O(S) words per look instead of O(b).
    struct alignas(kCacheLine) StreamOrder {
        std::atomic_flag launching = ATOMIC_FLAG_INIT;  // held around launch + push: list order == stream order
        std::atomic_flag polling = ATOMIC_FLAG_INIT;    // one dispatcher at a time walks a stream's list
        Ring<int> q;
    };
    struct alignas(kCacheLine) Running {
        int exec = -1;
        std::atomic<int> state{0};  // 0 idle, 1 in flight, 2 completion claimed by a polling dispatcher
        JobDesc job;
    };

    // Flag-polled completion: look at the oldest in-flight slot of every stream; whoever wins the 1 -> 2 claim runs
    // Algorithm 3, then the stream's next slot becomes the oldest.
    bool poll_flags() {
        bool any = false;
        for (int s = 0; s < S_; ++s) {
            StreamOrder& so = launched_[s];
            if (so.q.empty_approx()) continue;
            if (so.polling.test_and_set(std::memory_order_acquire)) continue;  // another dispatcher is on this stream
            int w;
            while (so.q.try_peek(w)) {
                Running& r = running_[w];
                if (r.state.load(std::memory_order_acquire) != 1) break;  // still being set up by the launching thread
                if (__atomic_load_n(&flags_[w * kFlagStride], __ATOMIC_ACQUIRE) == 0) break;
                int one = 1;
                if (!r.state.compare_exchange_strong(one, 2, std::memory_order_acq_rel)) break;
                int popped;
                so.q.try_pop(popped);
                on_complete(w);
                any = true;
            }
            so.polling.clear(std::memory_order_release);
        }
        return any;
    }

    // ---- Algorithm 2: FindJob -----------------------------------------------------------
    bool find_job(int w, Prepared& p, bool& stolen) {
        if (queues_[w].r.try_pop(p)) {  // local queue first: head of Q_w
            stolen = false;
            return true;
        }
        for (int k = 1; k < b_; ++k) {  // victim_id = (w_id + k) mod b, first job it meets
            int v = w + k;
            if (v >= b_) v -= b_;
            if (queues_[v].r.try_pop(p)) {  // try_steal == try_pop at the head
                stolen = true;
                return true;
            }
        }
        return false;
    }

    // ---- Algorithm 2: LaunchJob -------------------------------------------
    // Returns false if the job could not be taken by slot w after all (slot-bound executables): the caller releases w.
    bool launch_job(Prepared p, int w, bool stolen) {
        uint64_t t0 = now_ns();
        bool pinned = (p.home & kPinnedBit) != 0;
        const bool unbound = (p.home & kUnboundBit) != 0;  // bind-at-launch: nothing is tied to the executable yet
        int exec = p.exec;
        int rc = 0;
        if (stolen && slot_bound_.load(std::memory_order_acquire)) {
            int mine = -1;
            bool dummy = false;
            if (pinned || !free_execs_[w].r.try_pop(mine)) {
                // staged data lives with the victim's executable, or every executable of w is in a submitter's hands right
                // now: un-steal (there is room: the entry was just popped from that queue; jobs are independent, so order is free)
                queues_[p.home & ~(kPinnedBit | kUnboundBit)].r.push(p);
                n_queued_.fetch_add(1, std::memory_order_seq_cst);
                return false;
            }
            stats_.steals.fetch_add(1, std::memory_order_relaxed);
            rc = be_->bind(mine, w, p.job, &dummy);
            free_execs_[exec / epp_].r.push(exec);
            space_ec_.notify_all();
            exec = mine;
        } else if (stolen) {
            stats_.steals.fetch_add(1, std::memory_order_relaxed);
            int mine = -1;
            bool dummy = false;
            if (steal_policy_ == kSwap && !pinned && free_execs_[w].r.try_pop(mine)) {
                // The thief owns an exec that is already tied to M_w: give the job to it (only the
                // host-pointer copy nodes change) and hand the victim's exec back at once.
                rc = be_->bind(mine, w, p.job, &dummy);
                free_execs_[exec / epp_].r.push(exec);
                space_ec_.notify_all();
                exec = mine;
            } else {
                // JIT update retargets the victim's exec to read W_free's input memory, use
                // W_free's buffers and write W_free's output memory.
                rc = be_->bind(exec, w, p.job, &dummy);
            }
        } else if (unbound) {
            bool dummy = false;
            rc = be_->bind(exec, w, p.job, &dummy);  // the slot's own job: UpdateGraphParams now, on the launching thread
        }
        Running& r = running_[w];
        r.exec = exec;
        r.job = p.job;
        uint64_t inflight = inflight_.fetch_add(1, std::memory_order_seq_cst) + 1;
        if (own_poller_ && inflight == 1) poll_ec_.notify_all();  // the poller sleeps while nothing is in flight
        uint64_t hw = stats_.max_inflight.load(std::memory_order_relaxed);
        while (inflight > hw && !stats_.max_inflight.compare_exchange_weak(hw, inflight)) {
        }
        if (flags_) {  // clear the slot's completion word BEFORE it becomes visible as in flight
            __atomic_store_n(&flags_[w * kFlagStride], 0u, __ATOMIC_RELAXED);
            r.state.store(1, std::memory_order_release);
        }
        if (rc == 0) {
            if (flags_) {
                StreamOrder& so = launched_[w % S_];
                while (so.launching.test_and_set(std::memory_order_acquire)) cpu_relax();
                rc = be_->launch(exec, w, p.job);  // GraphLaunch
                if (rc == 0) so.q.push(w);         // room is guaranteed: at most b slots are in flight
                so.launching.clear(std::memory_order_release);
            } else {
                rc = be_->launch(exec, w, p.job);  // GraphLaunch + AddCallback
            }
        }
        stats_.launched.fetch_add(1, std::memory_order_relaxed);
        stats_.ns_launch.fetch_add(now_ns() - t0, std::memory_order_relaxed);
        if (rc != 0) {  // keep the books balanced so that drain returns; the error is sticky
            set_error(rc);
            int one = 1;
            if (!flags_ || r.state.compare_exchange_strong(one, 2, std::memory_order_acq_rel)) on_complete(w);
        }
        return true;
    }

    // ---- Algorithm 2: dispatcher main loop ----------------------------------------------
    // Dedicated completion thread (flag-polled mode): watch the words while anything is in flight, sleep otherwise.
    void poller_loop() {
        Backoff idle(4096);
        while (!stop_.load(std::memory_order_acquire)) {
            uint32_t seen = poll_ec_.prepare();
            if (poll_flags()) {
                idle = Backoff(4096);
                continue;
            }
            if (inflight_.load(std::memory_order_seq_cst) > 0) {
                idle.pause();
                continue;
            }
            if (stop_.load(std::memory_order_acquire)) break;
            poll_ec_.wait(seen, spin_ns_, kPollNs);  // woken by the launch that puts the first job in flight (or by stop)
            idle = Backoff(4096);
        }
    }

    void dispatcher_loop() {
        Backoff idle(4096);
        while (!stop_.load(std::memory_order_acquire)) {
            uint32_t seen = work_ec_.prepare();
            bool progressed = (flags_ && !own_poller_) ? poll_flags() : false;
            if (n_free_.load(std::memory_order_seq_cst) > 0 && n_queued_.load(std::memory_order_seq_cst) > 0) {
                int w;
                if (!pool_.try_pop(w)) {  // another dispatcher took it
                    idle.pause();
                    continue;
                }
                idle = Backoff(4096);
                n_free_.fetch_sub(1, std::memory_order_seq_cst);
                Prepared p;
                bool stolen = false;
                if (find_job(w, p, stolen)) {
                    n_queued_.fetch_sub(1, std::memory_order_seq_cst);
                    if (!launch_job(p, w, stolen)) {  // slot-bound executables and none of w's free: w goes back to the pool
                        pool_.push(w);
                        n_free_.fetch_add(1, std::memory_order_seq_cst);
                        idle.pause();
                    }
                } else {  // Alg. 2 l.7: no job -> the worker goes back to the pool
                    pool_.push(w);
                    n_free_.fetch_add(1, std::memory_order_seq_cst);
                }
                continue;
            }
            if (progressed) {
                idle = Backoff(4096);
                continue;
            }
            if (stop_.load(std::memory_order_acquire)) break;
            if (flags_ && !own_poller_ && inflight_.load(std::memory_order_seq_cst) > 0) {
                // Nobody will wake this thread when the GPU stores a flag: keep watching while work is in flight
                // (PAUSE for the first few thousand rounds, then yield between looks).
                idle.pause();
                continue;
            }
            // Sleep until there is both an idle worker and a queued job (or, polled mode, until a submit arrives).
            if (work_ec_.wait(seen, spin_ns_)) stats_.dispatcher_sleeps.fetch_add(1, std::memory_order_relaxed);
            idle = Backoff(4096);
        }
    }

    Backend* be_;
    volatile uint32_t* flags_ = nullptr;
    const int S_, b_, q_, epp_, steal_policy_;
    int active_ = 0;  // slots in service: b_ unless retire_slots() was called
    const uint64_t spin_ns_;
    std::unique_ptr<PaddedRing<Prepared>[]> queues_;
    std::unique_ptr<PaddedRing<int>[]> free_execs_;
    std::unique_ptr<Running[]> running_;
    std::unique_ptr<StreamOrder[]> launched_;
    Ring<int> pool_;
    alignas(kCacheLine) std::atomic<uint64_t> c_next_{0};
    alignas(kCacheLine) std::atomic<uint64_t> c_submitted_{0};
    alignas(kCacheLine) std::atomic<uint64_t> c_done_{0};
    alignas(kCacheLine) std::atomic<int64_t> n_queued_{0};
    alignas(kCacheLine) std::atomic<int64_t> n_free_{0};
    alignas(kCacheLine) std::atomic<int64_t> inflight_{0};
    EventCount work_ec_, space_ec_, done_ec_, poll_ec_;
    bool own_poller_ = false;
    std::atomic<bool> stop_{false};
    std::atomic<bool> slot_bound_{false};
    std::atomic<bool> lazy_bind_{false};
    std::atomic<int> err_{0};
    CoreStats stats_;
    std::vector<std::thread> dispatchers_;
};

}  // namespace setrt
