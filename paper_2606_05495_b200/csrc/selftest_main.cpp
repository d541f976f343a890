// selftest_main.cpp -- stand-alone driver of the host-only self tests (include/set.h "Host-only self tests"): the
// lock-free ring, FindJob's victim order and Algorithms 1-3 against a simulated device.  No CUDA call is made, so the
// program links without the CUDA runtime and can be built with -fsanitize=thread / -fsanitize=address:
//     python -m paper_2606_05495_b200.build --selftest thread     ->  paper_2606_05495_b200/build/selftest_thread
// Exit code 0 = every check passed (and the sanitizer reported nothing: TSAN_OPTIONS=halt_on_error=1 exitcode=66).
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <initializer_list>

#include "../../include/set.h"

int main(int argc, char** argv) {
    const int64_t scale = argc > 1 ? atoll(argv[1]) : 1;  // multiplies the job / token counts
    int bad = 0;
    for (int b : {1, 2, 5, 8, 64})
        for (int w = 0; w < b; ++w)
            for (uint64_t mask : {0ull, 1ull, ~0ull, 0x8000000000000001ull, 0x00f0ull}) {
                uint64_t m = b == 64 ? mask : mask & ((1ull << b) - 1);
                int want = -1;
                for (int k = 0; k < b && want < 0; ++k)
                    if (m >> ((w + k) % b) & 1) want = (w + k) % b;
                if (set_selftest_find_order(b, w, m) != want) ++bad;
            }
    printf("find_order: %s\n", bad ? "FAILED" : "ok");
    struct R { int cap, prod, cons; int64_t items; } rings[] = {{2, 1, 1, 20000}, {8, 3, 3, 20000}, {64, 4, 2, 20000}, {4, 2, 6, 5000}};
    for (auto& r : rings) {
        int64_t rc = set_selftest_ring(r.cap, r.prod, r.cons, r.items * scale);
        printf("ring cap=%d producers=%d consumers=%d items=%lld: %s (%lld)\n", r.cap, r.prod, r.cons, (long long)(r.items * scale),
               rc == 0 ? "ok" : "FAILED", (long long)rc);
        if (rc) ++bad;
    }
    // S, b, q, dispatchers, submitters, jobs, seed (bit 0: retarget steals, bit 1: flag-polled completion, bit 2: own poller thread, ...)
    struct S { int S, b, q, disp, subs; int64_t jobs; uint32_t seed; } scheds[] = {
        {4, 8, 2, 1, 1, 10000, 0}, {8, 32, 2, 1, 1, 10000, 1}, {8, 32, 2, 3, 2, 10000, 2}, {8, 32, 2, 2, 2, 10000, 3},
        {1, 1, 1, 1, 1, 1000, 3},  {4, 6, 1, 2, 3, 5000, 5},   {2, 64, 4, 2, 2, 10000, 4}, {8, 4096, 1, 1, 2, 20000, 2},
        {8, 32, 2, 1, 1, 10000, 6}, {8, 32, 2, 2, 2, 10000, 7}, {4, 8, 2, 1, 2, 10000, 6},   // bit 2: completion thread of its own
        {8, 32, 2, 1, 1, 10000, 14}, {8, 32, 2, 2, 2, 10000, 9}, {4, 8, 2, 1, 2, 10000, 10}, {8, 32, 2, 2, 1, 10000, 15},  // bit 3: bind at launch
        {8, 32, 2, 1, 1, 10000, 18}, {4, 32, 2, 2, 3, 10000, 22}, {8, 16, 2, 2, 2, 10000, 26},  // bit 4: slots beyond the streams retired, slot-bound
        {2, 4, 1, 1, 3, 10000, 32}, {8, 32, 2, 2, 2, 10000, 38}};  // bit 5: non-blocking submits that are retried
    for (auto& s : scheds) {
        uint64_t steals = 0;
        int64_t rc = set_selftest_scheduler(s.S, s.b, s.q, s.disp, s.subs, s.jobs * scale, s.seed, &steals);
        printf("scheduler S=%d b=%d q=%d dispatchers=%d submitters=%d jobs=%lld seed=%u: %s (%lld), %llu steals\n", s.S, s.b, s.q, s.disp,
               s.subs, (long long)(s.jobs * scale), s.seed, rc == 0 ? "ok" : "FAILED", (long long)rc, (unsigned long long)steals);
        if (rc) ++bad;
    }
    printf("%s\n", bad ? "SELFTEST FAILED" : "SELFTEST OK");
    return bad ? 1 : 0;
}
