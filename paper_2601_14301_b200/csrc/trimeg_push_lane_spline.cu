// trimeg_push_lane_spline.cu -- push_lane_kernel compiled for row f3's own case alone (ring x sector mesh, field on cubic
// B-spline planes, rigorous equations, analytic equilibrium): see TRIMEG_SPLINE_ONLY in trimeg_device.cuh.
// launch_push_lane_spline().
#define TRIMEG_SPLINE_ONLY 1
#include "trimeg_push_lane.cu"
