// Driver for tests/test_oracle_sanitizers.py: the host-side schedule builder of the Cholesky task graph
// (paper_1608_04329_b200/csrc/chol_schedule.cu is plain C++: compiled here by g++ as one translation unit) under
// AddressSanitizer + UndefinedBehaviorSanitizer over a range of (tile rows, super-block, CTA count).
#include "../../paper_1608_04329_b200/csrc/chol_schedule.cu"
#include <cstdio>

int main() {
  long long tasks = 0;
  const int nts[] = {1, 2, 3, 5, 8, 16, 21, 32, 63, 100};
  const int Ks[] = {1, 2, 3, 7, 16, 48, 104, 148};
  for (int nt : nts)
    for (int K : Ks) {
      if ((long long)K > (long long)nt * nt) continue;
      const int sb = nt <= 20 ? nt : 8;
      const hsp::CholSchedule s = hsp::chol_build_schedule(nt, sb, K);
      if ((int)s.list_off.size() != K + 1 || s.list_off[K] != (int)s.tasks.size() || !(s.makespan_us > 0.0)) { std::printf("FAILED nt=%d K=%d\n", nt, K); return 1; }
      tasks += (long long)s.tasks.size();
    }
  std::printf("ok %lld tasks\n", tasks);
  return 0;
}
