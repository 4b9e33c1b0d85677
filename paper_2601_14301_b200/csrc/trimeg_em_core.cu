// trimeg_em_core.cu -- rhs_em_kernel compiled for the core case alone (ring x sector mesh, harmonic field, rigorous equations,
// analytic equilibrium): see TRIMEG_CORE_ONLY in trimeg_device.cuh.  launch_rhs_em_core().
#define TRIMEG_CORE_ONLY 1
#include "trimeg_em.cu"
