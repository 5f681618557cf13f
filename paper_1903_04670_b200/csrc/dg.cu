// dg.cu -- dgfs_step / dgfs_advect_rhs (placeholder until the DG transport kernels land).
#include "ctx.h"
using namespace dgfs;
extern "C" int dgfs_step(dgfs_ctx* c, const dgfs_mesh1d*, double*, double, int, void*) {
  if (!c) return DGFS_EINVAL;
  return set_error(c, DGFS_ENOSUP, "dgfs_step: not implemented yet");
}
extern "C" int dgfs_advect_rhs(dgfs_ctx* c, const dgfs_mesh1d*, const double*, double*, void*) {
  if (!c) return DGFS_EINVAL;
  return set_error(c, DGFS_ENOSUP, "dgfs_advect_rhs: not implemented yet");
}
