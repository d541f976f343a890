// set_ring.hpp -- bounded lock-free multi-producer / multi-consumer ring.
//
// Used for the three host-side structures of the method:
//   Q_w     per-slot job queue of prepared graph executables
//   W_pool  free worker pool, filled only by completion callbacks
//   exec free lists (the "bounded pool of cudaGraphExec instances" of BASELINE.json:north_star)
//
// The paper's queues are "thread-safe" without saying how and blames a global mutex
// for the queue model's cost; here every queue is a ring with one sequence number per
// cell, so producers (submitter threads, the driver's callback thread) and consumers (dispatcher
// threads, owner pop and thief steal alike) never take a lock.  try_pop and try_steal are the same
// operation: both take the OLDEST entry ("the head of Q_free is popped", "steal the first
// job it meets").  The owner/thief asymmetry of a Chase-Lev deque does not apply because the producer
// (submitter) and the consumer (dispatcher) are different threads (SURVEY.md §7 "Hard parts").
#pragma once
#include <atomic>
#include <cstddef>
#include <cstdint>
#include <memory>
#include <new>

#include <sched.h>

namespace setrt {

constexpr size_t kCacheLine = 64;

// Spin politely: PAUSE for the first `spins` rounds, then give the core away each round, so that a waiter never
// starves the thread it is waiting for when there are fewer cores than threads.
struct Backoff {
    explicit Backoff(int spins = 128) : left(spins) {}
    void pause() {
        if (left > 0) {
            --left;
#if defined(__x86_64__) || defined(__i386__)
            __builtin_ia32_pause();
#else
            asm volatile("" ::: "memory");
#endif
        } else {
            sched_yield();
        }
    }
    int left;
};

template <typename T>
class Ring {
    struct alignas(16) Cell {
        std::atomic<uint64_t> seq;
        T value;
    };

  public:
    Ring() = default;
    explicit Ring(size_t capacity) { init(capacity); }
    Ring(const Ring&) = delete;
    Ring& operator=(const Ring&) = delete;

    // capacity is rounded up to a power of two >= 2
    void init(size_t capacity) {
        size_t cap = 2;
        while (cap < capacity) cap <<= 1;
        mask_ = cap - 1;
        cells_.reset(new Cell[cap]);
        for (size_t i = 0; i < cap; ++i) cells_[i].seq.store(i, std::memory_order_relaxed);
        head_.store(0, std::memory_order_relaxed);
        tail_.store(0, std::memory_order_relaxed);
    }

    size_t capacity() const { return mask_ + 1; }

    bool try_push(const T& v) {
        uint64_t pos = tail_.load(std::memory_order_relaxed);
        for (;;) {
            Cell& c = cells_[pos & mask_];
            uint64_t seq = c.seq.load(std::memory_order_acquire);
            int64_t dif = (int64_t)seq - (int64_t)pos;
            if (dif == 0) {
                if (tail_.compare_exchange_weak(pos, pos + 1, std::memory_order_relaxed)) {
                    c.value = v;
                    c.seq.store(pos + 1, std::memory_order_release);
                    return true;
                }
            } else if (dif < 0) {
                return false;  // full
            } else {
                pos = tail_.load(std::memory_order_relaxed);
            }
        }
    }

    // For pushes that are logically guaranteed room (the entry count is bounded below the capacity by the
    // caller's own accounting).  try_push can still report "full" for a moment: a consumer that claimed the
    // cell one lap earlier may have been preempted between its head_ CAS and its seq store.  That state is
    // transient, so wait it out instead of dropping the entry.
    void push(const T& v) {
        Backoff bo;
        while (!try_push(v)) bo.pause();
    }

    bool try_pop(T& out) {
        uint64_t pos = head_.load(std::memory_order_relaxed);
        for (;;) {
            Cell& c = cells_[pos & mask_];
            uint64_t seq = c.seq.load(std::memory_order_acquire);
            int64_t dif = (int64_t)seq - (int64_t)(pos + 1);
            if (dif == 0) {
                if (head_.compare_exchange_weak(pos, pos + 1, std::memory_order_relaxed)) {
                    out = c.value;
                    c.seq.store(pos + mask_ + 1, std::memory_order_release);
                    return true;
                }
            } else if (dif < 0) {
                return false;  // empty
            } else {
                pos = head_.load(std::memory_order_relaxed);
            }
        }
    }

    // Look at the oldest entry without taking it.  Only meaningful while the caller is the ring's sole consumer
    // (producers may push concurrently): used for the per-stream launch-order lists the polling dispatcher walks.
    bool try_peek(T& out) const {
        const uint64_t pos = head_.load(std::memory_order_relaxed);
        const Cell& c = cells_[pos & mask_];
        if (c.seq.load(std::memory_order_acquire) != pos + 1) return false;
        out = c.value;
        return true;
    }

    // Racy size estimate (exact when quiescent).
    size_t size_approx() const {
        uint64_t t = tail_.load(std::memory_order_relaxed), h = head_.load(std::memory_order_relaxed);
        return t >= h ? (size_t)(t - h) : 0;
    }
    bool empty_approx() const { return size_approx() == 0; }

  private:
    alignas(kCacheLine) std::atomic<uint64_t> head_{0};
    alignas(kCacheLine) std::atomic<uint64_t> tail_{0};
    alignas(kCacheLine) size_t mask_ = 0;
    std::unique_ptr<Cell[]> cells_;
};

}  // namespace setrt
