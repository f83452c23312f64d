// parallel_for.h -- plan-time host work is independent per channel (and per chunk): fn(i) for i in [0, n) on
// the host cores.  No CUDA in here (tests/host_parallel_check.cpp builds it with g++).
//
// The callers are extern "C" entry points, so nothing may leave a worker thread as an exception (that is
// std::terminate) and a thread that cannot be created must not take the process down either:
//   - a worker that throws (std::bad_alloc from a growing table) stops the loop for everyone; after the
//     join the failure is re-thrown as std::bad_alloc in the CALLING thread, where the entry point's handler
//     turns it into BLINK_ENOMEM -- the same place a serial loop would have failed;
//   - if std::thread cannot start (std::system_error), the indices that are left run on the threads that
//     did start and on the calling thread, which always takes part.
#pragma once

#include <algorithm>
#include <atomic>
#include <new>
#include <thread>
#include <vector>

namespace blink {
template <class F> inline void parallel_for(int n, F fn, int max_threads = 32) {
  const int hw = (int)std::thread::hardware_concurrency();
  const int nt = std::min(n, std::max(1, std::min(hw, max_threads)));
  std::atomic<int> next{0};
  std::atomic<bool> failed{false};
  auto work = [&]() noexcept {
    try {
      for (;;) {
        const int i = next.fetch_add(1);
        if (i >= n || failed.load(std::memory_order_relaxed)) break;
        fn(i);
      }
    } catch (...) {
      failed.store(true);
    }
  };
  std::vector<std::thread> th;
  try {
    th.reserve(nt > 1 ? nt - 1 : 0);
    for (int t = 1; t < nt; ++t) th.emplace_back(work);
  } catch (...) {
    // fewer helpers than wanted, or none: what is left runs below
  }
  work();
  for (auto &x : th) x.join();
  if (failed.load()) throw std::bad_alloc();
}
}  // namespace blink
