// trimeg_mesh.cuh -- vertex and triangle numbering of the ring x sector mesh (reading O1), host and device.
#pragma once
#include <cuda_runtime.h>

namespace trimeg {

__host__ __device__ __forceinline__ int vertex_id(int n_theta, int i, int j)
{   // v(i, j) = 1 + (i-1) n_theta + (j mod n_theta), i >= 1
    if (j >= n_theta) j -= n_theta;
    return 1 + (i - 1) * n_theta + j;
}
// tri != NULL: unstructured mesh (row f4), the vertex triples come from the table [n_tri][3]
__host__ __device__ __forceinline__ void tri_vertices(int n_theta, const int *tri, int t, int v[3])
{
    if (tri) { v[0] = tri[3 * (size_t)t]; v[1] = tri[3 * (size_t)t + 1]; v[2] = tri[3 * (size_t)t + 2]; return; }
    if (t < n_theta) { v[0] = 0; v[1] = vertex_id(n_theta, 1, t); v[2] = vertex_id(n_theta, 1, t + 1); return; }
    const int u = t - n_theta, k = u & 1, c = u >> 1, i = c / n_theta + 1, j = c % n_theta;
    v[0] = vertex_id(n_theta, i, j);
    if (k == 0) { v[1] = vertex_id(n_theta, i + 1, j); v[2] = vertex_id(n_theta, i + 1, j + 1); }
    else { v[1] = vertex_id(n_theta, i + 1, j + 1); v[2] = vertex_id(n_theta, i, j + 1); }
}

}  // namespace trimeg
