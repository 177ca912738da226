// placeholder: tables not built yet -> the direct kernel is used
#include "mdsm_internal.h"
int mdsm_tiled_build_tables(mdsm_plan *p) { p->tiled_f32.ok = false; p->tiled_u8.ok = false; return MDSM_OK; }
void mdsm_tiled_free_tables(mdsm_plan *) {}
int mdsm_launch_dedisperse_tiled(mdsm_plan *, const void *, int, int, int, void *, cudaStream_t)
{
    mdsm_set_error("tiled kernel not built");
    return MDSM_EINVAL;
}
