// grid.cuh -- geometry of the padded structure-of-arrays state in HBM and the small device control block.
//
// Layout: every field is one padded 3-D array [npz][npy][sx], x fastest;
// np = n + 2g on active axes (g = 3 / 4 / 2), np = n on inactive ones; the row pitch sx rounds npx up
// to 16 bytes and the field stride fs rounds sx*npy*npz up to 256 bytes, so that every row start is
// 16-byte aligned.  A state is five such arrays (E, Mx, My, Mz, R); the generic kernel keeps another seven
// (v_x, v_y, v_z, p, a_x, a_y, a_z).  Only face ghosts are ever filled or read: the sweeps are
// dimension-by-dimension, so edge and corner ghosts stay zero and are never used.
#pragma once
#include <cuda_runtime.h>

namespace hydro {

struct Geom {
    int n[3];        // interior extents nx, ny, nz
    int g[3];        // ghost width per axis (0 when inactive)
    int np[3];       // padded extents
    long long sx;    // row pitch in elements
    long long sxy;   // plane pitch = sx * np[1]
    long long fs;    // field stride in elements
    __host__ __device__ long long pidx(int i, int j, int k) const {  // i,j,k interior-relative
        return (long long)(k + g[2]) * sxy + (long long)(j + g[1]) * sx + (i + g[0]);
    }
};

// Device-resident step control: current time, current dt, the max signal speed of the state at the start
// of the step (as the bit pattern of a non-negative double, so that atomicMax on integers orders it)
// and the sticky unphysical flag (reading Q16).
struct Ctl {
    double t;
    double dt;
    unsigned long long maxspeed_bits;
    int flag;
    int pad;
    unsigned long long maxspeed_next_bits;  // max speed of the state the running step is producing (stage-3 epilogue)
};

struct HubbleParams {  // closed-form ghost fill (readings Q13, Q14)
    double origin[3];
    double t0, e0, n0;
    double b[3];
    double dx;
};

}  // namespace hydro
