// trimeg_push_lane_core.cu -- push_lane_kernel compiled for the core case alone (ring x sector mesh, harmonic field, rigorous
// equations): see TRIMEG_CORE_ONLY in trimeg_device.cuh.  launch_push_lane_core().
#define TRIMEG_CORE_ONLY 1
#include "trimeg_push_lane.cu"
