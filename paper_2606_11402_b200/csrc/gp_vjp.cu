// placeholder, replaced below
#include "gp_cond.cuh"
namespace gp {
gp_status run_vjp(const OpCtx&, const void*, const void*, const void*, void*, double*) { return GP_ERR_UNSUPPORTED; }
gp_status head_vjp(const OpCtx&, const void*, const void*, void*, double*) { return GP_ERR_UNSUPPORTED; }
}
