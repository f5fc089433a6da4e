// loc_spectra.cu -- spectral-line map kernel.  Placeholder until the map kernels land.
#include <stdio.h>

#include "loc_internal.cuh"

int loc_launch_spectra(loc_model *m, int trans, const double *dir, int nx, int ny, const int64_t *aff, const double *offsets_cm,
                       float *dev_out)
{
    snprintf(m->err, sizeof(m->err), "loc_spectra: not implemented yet");
    return LOC_ESTATE;
}
