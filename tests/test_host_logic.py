"""Host-side logic of the scheduler, exercised without a GPU through the library's self-test entry points:
the lock-free ring, FindJob's steal order (Alg. 2 l.8-17) and Algorithms 1-3 end to end
against a simulated device."""
import random

import pytest


def test_find_order_matches_algorithm2(libset):
    rng = random.Random(7)
    for b in (1, 2, 5, 8, 32, 64):
        for _ in range(200):
            w = rng.randrange(b)
            mask = rng.getrandbits(b) if rng.random() < 0.8 else 0
            # Alg. 2: own queue first, else victim = (w + k) mod b for k = 1..b-1, else NULL
            want = -1
            if mask >> w & 1:
                want = w
            else:
                for k in range(1, b):
                    v = (w + k) % b
                    if mask >> v & 1:
                        want = v
                        break
            assert libset.selftest_find_order(b, w, mask) == want
    assert libset.selftest_find_order(8, 3, 0b00000110) == 1      # wraps around: 4..7 empty, then 0 empty, then 1
    assert libset.selftest_find_order(8, 8, 1) == -2              # w out of range


@pytest.mark.parametrize("cap,prod,cons,items", [(2, 1, 1, 20000), (8, 3, 3, 30000), (64, 4, 2, 30000), (4, 2, 6, 10000)])
def test_ring_delivers_every_token_exactly_once(libset, cap, prod, cons, items):
    assert libset.selftest_ring(cap, prod, cons, items) == 0


@pytest.mark.parametrize("S,b,q,disp,subs,jobs,seed", [
    (4, 8, 2, 1, 1, 20000, 0),      # config 0/2/3 geometry, swap steals
    (8, 32, 2, 1, 1, 30000, 1),     # config 1/4 geometry, retarget steals (odd seed)
    (8, 32, 2, 3, 2, 30000, 2),     # several dispatchers and submitters
    (1, 1, 1, 1, 1, 2000, 3),       # degenerate: one worker
    (4, 6, 1, 2, 3, 10000, 5),      # max_inflight not a multiple of the stream count -> rounded up
    (2, 64, 4, 2, 2, 20000, 4),
    (8, 32, 2, 1, 1, 20000, 16 + 2),    # a loop pipeline's geometry: slots 8..31 retired, executables bound to their slot
    (4, 32, 2, 2, 3, 20000, 16 + 4),    # the same with a completion thread, several dispatchers and submitters
    (8, 8, 2, 1, 1, 5000, 16),          # nothing to retire
    (2, 4, 1, 1, 3, 20000, 32),         # non-blocking submits (set_try_submit_dims) retried by three submitters against 4 slots
    (8, 32, 2, 2, 2, 20000, 32 + 4 + 2),
])
def test_scheduler_algorithms_on_simulated_device(libset, S, b, q, disp, subs, jobs, seed):
    rc, steals = libset.selftest_scheduler(S, b, q, disp, subs, jobs, seed)
    assert rc == 0
    assert steals >= 0


def test_scheduler_zero_jobs_and_bad_args(libset):
    rc, _ = libset.selftest_scheduler(4, 8, 2, 1, 1, 0, 0)
    assert rc == 0
    rc, _ = libset.selftest_scheduler(0, 8, 2, 1, 1, 10, 0)
    assert rc == -1


def test_scheduler_core_is_clean_under_thread_sanitizer():
    """The lock-free ring and Algorithms 1-3 (set_core.hpp, set_ring.hpp) built with -fsanitize=thread and run against the
    simulated device: no data race reported (TSAN exit code 66), every check passed (exit code 0)."""
    import os
    import subprocess
    from paper_2606_05495_b200 import build as b
    exe = b.build_selftest("thread")
    r = subprocess.run([exe, "1"], capture_output=True, text=True, timeout=600,
                       env=dict(os.environ, TSAN_OPTIONS="halt_on_error=0 exitcode=66"))
    assert "SELFTEST OK" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]
    assert r.returncode == 0 and "WARNING: ThreadSanitizer" not in r.stderr, r.stderr[-3000:]


def test_divide_by_nine_multiplier_is_exact_on_the_mean_filters_range():
    """K18 (set_k_mean3x3_u8) divides the 3 x 3 sum (at most 9 * 255) by 9 as (v * 7282) >> 16 in each 16-bit half."""
    assert all((v * 7282) >> 16 == v // 9 for v in range(9 * 255 + 1))
