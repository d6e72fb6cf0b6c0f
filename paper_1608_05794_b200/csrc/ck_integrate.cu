// Workspace sizing (include/ck.h: ck_workspace_bytes).
#include "ck_internal.h"
using namespace ck;

size_t ck_ros_workspace(const ck_mech* m, int64_t n);
size_t ck_rkf_workspace(const ck_mech* m, int64_t n);
size_t ck_jac_workspace(const ck_mech* m, int64_t n);

extern "C" int32_t ck_workspace_bytes(const ck_mech* m, int32_t op, int64_t n, size_t* bytes) {
  if (!m || !bytes || n < 0 || (op != CK_OP_ROS && op != CK_OP_RKF45 && op != CK_OP_JAC)) { set_error("ck_workspace_bytes: bad argument"); return CK_EINVAL; }
  *bytes = (op == CK_OP_ROS) ? ck_ros_workspace(m, n) : (op == CK_OP_RKF45 ? ck_rkf_workspace(m, n) : ck_jac_workspace(m, n));
  return CK_OK;
}
