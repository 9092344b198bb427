// kernel_lattice.cuh -- part of vox.cu (included there, once): K0 of the fused lattice path (vertex-plane slabs + packed vertex copy).
#pragma once

// ------------------------------------------------------------------------------------------
// K0 (fused lattice path): one pass over the lattice vertices that
//  (1) records per mesh, axis and vertex plane of the lattice the largest coordinate and the largest
//      (extent - coordinate) over the plane's vertices.  From these a tile finds the index range of the cells whose
//      tets can reach it (k4_flat<.., LATTICE>) -- no per-tet bbox search, no pair list;
//        slab of mesh m: [x: lo'(cx+1) hi(cx+1) | y: lo'(cy+1) hi(cy+1) | z: lo'(cz+1) hi(cz+1)],  lo' = extent - min
//      (zero-initialised by the memset of the header; coordinates lie in [0, extent], so a plain max suffices);
//  (2) writes a 16-byte copy (x, y, z, 0) of every vertex: K4 then gathers a vertex with one LDG.128 instead of three
//      4-byte loads (the gather is what loads the LSU pipe in K4's setup, profiles/r02).
// One CTA per (x plane i, chunk of y rows, mesh); its warps take the chunk's rows in turn, lanes run along z.
// x: registers + warp reduce; y: warp reduce per row; z: shared-memory atomics; one global atomicMax per value and CTA.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k0_slabs(const int32_t* __restrict__ verts, int cx, int cy, int cz, int ex, int ey,
                                                int ez, int jchunk, int* __restrict__ slab, int4* __restrict__ verts4) {
    extern __shared__ int s_z[];  // [cz+1] lo', [cz+1] hi
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = blockIdx.x, m = blockIdx.z;
    const int j0 = blockIdx.y * jchunk, j1 = min(cy + 1, j0 + jchunk);
    int* sl = slab + (size_t)m * 2 * (cx + cy + cz + 3);
    int* xlo = sl, *xhi = sl + cx + 1, *ylo = sl + 2 * (cx + 1), *yhi = ylo + cy + 1, *zlo = ylo + 2 * (cy + 1), *zhi = zlo + cz + 1;
    for (int k = tid; k < 2 * (cz + 1); k += 256) s_z[k] = 0;
    __syncthreads();
    int mxlo = 0, mxhi = 0;
    for (int j = j0 + warp; j < j1; j += 8) {
        int mylo = 0, myhi = 0;
        const size_t v0 = (((size_t)m * (cx + 1) + i) * (cy + 1) + j) * (size_t)(cz + 1);
        const int32_t* row = verts + 3 * v0;
        for (int k = lane; k <= cz; k += 32) {
            const int x = __ldg(row + 3 * k), y = __ldg(row + 3 * k + 1), z = __ldg(row + 3 * k + 2);
            VOX_CHECK(v0 + k < (size_t)gridDim.z * (cx + 1) * (cy + 1) * (cz + 1), CK_K0_VERT);
            verts4[v0 + k] = make_int4(x, y, z, 0);
            mxhi = max(mxhi, x); mxlo = max(mxlo, ex - x);
            myhi = max(myhi, y); mylo = max(mylo, ey - y);
            atomicMax(s_z + k, ez - z);
            atomicMax(s_z + cz + 1 + k, z);
        }
        myhi = __reduce_max_sync(0xFFFFFFFFu, myhi);
        mylo = __reduce_max_sync(0xFFFFFFFFu, mylo);
        if (lane == 0) { atomicMax(yhi + j, myhi); atomicMax(ylo + j, mylo); }
    }
    mxhi = __reduce_max_sync(0xFFFFFFFFu, mxhi);
    mxlo = __reduce_max_sync(0xFFFFFFFFu, mxlo);
    if (lane == 0) { atomicMax(xhi + i, mxhi); atomicMax(xlo + i, mxlo); }
    __syncthreads();
    for (int k = tid; k <= cz; k += 256) { atomicMax(zlo + k, s_z[k]); atomicMax(zhi + k, s_z[cz + 1 + k]); }
}
