// igr_rhs_tile.cuh -- interface of the tiled RHS kernel (row a4, optionally fused with a5/a6).
#pragma once
#include <cuda.h>
#include "igr_common.cuh"

struct RhsTileMaps {
    CUtensorMap q[3];      // 4-D maps (x, y, z, field) of the three state buffers
    CUtensorMap sig[2];    // 3-D maps of the two Sigma buffers
    bool valid;
};

struct RhsTileArgs {
    float *r[5];           // unfused: RHS out (fp32, padded)
    const void *qn[5];     // fused: q^n (pointwise read)
    void *qout[5];         // fused: new stage state (pointwise write)
    float beta, dt;        // fused: q_out = q_n + beta ((q_s - q_n) + dt r)
    int read_qn;           // fused: 0 in stage 1 (q_n == q_s, taken from the tile)
    WaveResult *wave;      // fused stage 3: wave speed of q_out (may be NULL)
    float gamma, inv_dx;
    int zc;                // planes per z-chunk
};

// returns 0 on success, else a CUresult/cudaError-like code (message in `err`)
int rhs_tile_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state,
                       void *const sig[2], RhsTileMaps *out, const char **err);
// order: 5 or 3; fused: epilogue performs the RK update instead of storing r
void launch_rhs_tile(const Grid &g, int storage, int order, bool fused, const CUtensorMap &qmap,
                     const CUtensorMap &smap, RhsTileArgs a, cudaStream_t st);
int rhs_tile_default_zc(const Grid &g);
