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
    float *r[7];           // unfused: RHS out (fp32, padded); 5 fields, or 7 with two fluids
    const void *qn[7];     // fused: q^n (pointwise read)
    void *qout[7];         // fused: new stage state (pointwise write)
    float beta, dt;        // fused: q_out = q_n + beta ((q_s - q_n) + dt r)
    int read_qn;           // fused: 0 in stage 1 (q_n == q_s, taken from the tile)
    WaveResult *wave;      // fused stage 3: wave speed of q_out (may be NULL)
    float gamma, inv_dx;
    int zc;                // planes per z-chunk
    int nf;                // 5 (default when 0), or 7: two fluids (reading A21)
    float k1, k2;          // two fluids: 1/(gamma_1 - 1), 1/(gamma_2 - 1)
};

// returns 0 on success, else a CUresult/cudaError-like code (message in `err`)
int rhs_tile_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state,
                       void *const sig[2], int nf, RhsTileMaps *out, const char **err);
// order: 5 or 3; fused: epilogue performs the RK update instead of storing r
void launch_rhs_tile(const Grid &g, int storage, int order, bool fused, const CUtensorMap &qmap,
                     const CUtensorMap &smap, RhsTileArgs a, cudaStream_t st);
int rhs_tile_default_zc(const Grid &g);
