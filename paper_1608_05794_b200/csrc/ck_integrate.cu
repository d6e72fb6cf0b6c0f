// Integrators (placeholder translation unit while the step-attempt kernels are brought up).
#include "ck_internal.h"
using namespace ck;

extern "C" int32_t ck_workspace_bytes(const ck_mech* m, int32_t op, int64_t n, size_t* bytes) {
  if (!m || !bytes || n < 0 || (op != CK_OP_ROS && op != CK_OP_RKF45)) { set_error("ck_workspace_bytes: bad argument"); return CK_EINVAL; }
  *bytes = 256;
  return CK_OK;
}
extern "C" int32_t ck_jac(const ck_mech*, int64_t, const double*, int64_t, const double*, int32_t, double, double, double,
                          double*, int64_t, void*) { set_error("ck_jac: not built yet"); return CK_EUNSUPPORTED; }
extern "C" int32_t ck_integrate_ros(const ck_mech*, int64_t, double*, int64_t, const double*, double, const ck_opts*, int32_t*,
                                    int32_t*, int32_t*, double*, void*, size_t, ck_report*, void*) { set_error("ck_integrate_ros: not built yet"); return CK_EUNSUPPORTED; }
extern "C" int32_t ck_integrate_rkf45(const ck_mech*, int64_t, double*, int64_t, const double*, double, const ck_opts*, int32_t*,
                                      int32_t*, int32_t*, double*, void*, size_t, ck_report*, void*) { set_error("ck_integrate_rkf45: not built yet"); return CK_EUNSUPPORTED; }
