// Device-side counters of the integrators (first 256 bytes of the caller's workspace) and the host-side
// report assembly shared by ck_integrate_ros / ck_integrate_rkf45.
#pragma once
#include <vector>

#include "ck_internal.h"

namespace ck {

struct DevStats {
  unsigned long long queue;        // work-queue head (next reactor to hand out)
  unsigned long long attempts, accepted, rejected, rhs_evals, jac_evals, failed;
  unsigned long long lane_active;  // lane-slots that did useful work in the step-attempt loop
  unsigned long long lane_total;   // lane-slots issued
  unsigned long long n_evicted;    // reactors the capped classification phase hands on to the resumed thread-per-reactor phase
  unsigned long long queue2;       // work-queue head of the finisher
  unsigned long long qempty;       // set once the main queue ran dry
  unsigned long long n_evicted_m;  // RKF45 classification: reactors of the middle class (narrow finisher, started at once;
                                   // listed from the back of the second eviction list)
  unsigned long long queue_m;      // work-queue head of that finisher
  unsigned long long sum_pred[3];  // predicted remaining attempts summed per class: 0 resumed, 1 middle, 2 stragglers
  unsigned long long spare[3];
  unsigned long long n_evicted_b;  // ... of which predicted stragglers (handed to the wide low-latency finisher; listed from
                                   // the back of the eviction list)
  unsigned long long queue_b;      // work-queue head of the wide finisher
  unsigned long long n_evicted_n;  // reactors handed to the narrow (throughput) finisher at the end-game
  unsigned long long queue_c;      // work-queue head of the resumed thread-per-reactor phase
  unsigned long long pad[8];
};
static_assert(sizeof(DevStats) == 256, "DevStats is the 256-byte header of the workspace");

// mean over work units of Eq. 20 at width P for the static linear reactor->lane mapping
inline double waste_static(const std::vector<int>& attempts, int P) {
  const size_t n = attempts.size();
  if (n == 0) return 0.0;
  double sum = 0.0;
  size_t units = 0;
  for (size_t b = 0; b < n; b += P) {
    long long tot = 0;
    int mx = 0;
    const size_t e = std::min(n, b + P);
    for (size_t i = b; i < e; ++i) { tot += attempts[i]; mx = std::max(mx, attempts[i]); }
    if (mx > 0) sum += 1.0 - (double)tot / ((double)(e - b) * mx);
    units++;
  }
  return sum / (double)units;
}

}  // namespace ck
