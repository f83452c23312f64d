// Host-side check of paper_2405_13478_b200/csrc/parallel_for.h (built and run by tests/test_host_logic.py,
// CPU only): every index runs exactly once whatever the thread count, and a worker that throws does not
// end the process (an exception leaving a std::thread is std::terminate) -- the failure comes back in the
// calling thread as std::bad_alloc, which the C entry points turn into BLINK_ENOMEM.  Prints "OK" or "FAIL ...".
#include <cstdio>
#include <stdexcept>
#include <vector>

#include "../paper_2405_13478_b200/csrc/parallel_for.h"

int main() {
  for (int threads : {1, 2, 8, 32}) {
    for (int n : {0, 1, 7, 1000}) {
      std::vector<std::atomic<int>> hit(n > 0 ? n : 1);
      for (auto &h : hit) h.store(0);
      blink::parallel_for(n, [&](int i) { hit[i].fetch_add(1); }, threads);
      for (int i = 0; i < n; ++i)
        if (hit[i].load() != 1) { std::printf("FAIL index %d ran %d times (n %d, threads %d)\n", i, hit[i].load(), n, threads); return 1; }
    }
    bool caught = false;
    std::atomic<int> ran{0};
    try {
      blink::parallel_for(500, [&](int i) {
        ran.fetch_add(1);
        if (i == 3) throw std::bad_alloc();
        if (i == 4) throw std::runtime_error("any exception type");
      }, threads);
    } catch (const std::bad_alloc &) {
      caught = true;
    }
    if (!caught) { std::printf("FAIL a throwing body was not reported (threads %d)\n", threads); return 1; }
    if (ran.load() < 1 || ran.load() > 500) { std::printf("FAIL ran %d\n", ran.load()); return 1; }
  }
  std::printf("OK\n");
  return 0;
}
