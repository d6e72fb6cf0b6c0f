// Declarations shared by the two ROS4 drivers: the fused CTA-per-reactor kernel (ck_ros.cu) and the batched rounds
// (ck_ros_rounds.cu).
#pragma once
#include "ck_internal.h"
#include "ck_stats.h"

namespace ck {

namespace ros4c {  // Table C.3
constexpr double gam = 0.57282;
constexpr double a21 = 2.0, a31 = 1.867943637803922, a32 = 0.2344449711399156;
constexpr double c21 = -7.137615036412310, c31 = 2.580708087951457, c32 = 0.6515950076447975;
constexpr double c41 = -2.137148994382534, c42 = -0.3214669691237626, c43 = -0.6949742501781779;
constexpr double m1 = 2.255570073418735, m2 = 0.2870493262186792, m3 = 0.4353179431840180, m4 = 1.093502252409163;
constexpr double e1 = -0.2815431932141155, e2 = -0.07276199124938920, e3 = -0.1082196201495311, e4 = -1.093502252409163;
}  // namespace ros4c

struct RosArgs {
  long long n, ld;
  double* y;
  const double* p;
  double dt, rtol, atol, h0;
  int jac_mode, max_steps, use_queue;
  int *n_accept, *n_reject, *status;
  double* h_last;
  int* att;  // [n] attempts per reactor (workspace; feeds the waste metric)
  DevStats* stats;
  // resume mode (tail of the batched rounds): reactors list[0 .. *list_n) continue from the state the rounds left
  const int* list;
  const int* list_n;
  const double *rt, *rh, *rfac;   // [n] time reached, next step size, fac_max
  const int *racc, *rrej;         // [n] accepted / rejected attempts so far
};

// launch the fused kernel on `st` (grid sized for n_hint reactors); defined in ck_ros.cu
int32_t ros_fused_launch(const ck_mech* m, const RosArgs& a, long long n_hint, int* G_used, cudaStream_t st);
size_t ros_fused_workspace(int64_t n);

// batched rounds (ck_ros_rounds.cu)
bool ros_rounds_supported(const ck_mech* m);
size_t ros_rounds_workspace(const ck_mech* m, int64_t n);
int32_t ros_rounds_run(const ck_mech* m, int64_t n, double* y, int64_t ld, const double* p, double dt, const ck_opts* o,
                       int32_t* n_accept, int32_t* n_reject, int32_t* status, double* h_last, void* ws, size_t ws_bytes,
                       int* rounds, double* lane_util, cudaStream_t st);

}  // namespace ck
