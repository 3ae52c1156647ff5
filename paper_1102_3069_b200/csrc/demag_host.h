// demag_host.h -- host-side demagnetisation kernel set-up (see demag_host.cpp).
#pragma once
#include <cstddef>
#include <string>

namespace mmh {

// Real-space cell-averaged tensor (xx,yy,zz,xy,xz,yz) at n integer cell offsets, images summed.
void tensor_at(const double cell[3], const int grid[3], const int pbc[3], size_t n, const long* off,
               double* out);

// Transformed kernel, one octant: khat_out[6][C2][C1][C0] float32, C = P/2+1, includes -1/(P0 P1 P2).
// Returns 0, or an mm_status value (2 = out of memory, 5 = unsupported size) with a message in *err.
int build_khat(const double cell[3], const int grid[3], const int pbc[3], float* khat_out,
               std::string* err);

}  // namespace mmh
