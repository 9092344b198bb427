// kernel_tile_k4.cuh -- part of vox.cu (included there, once): the K4 kernel k4_flat (binned and fused-lattice instantiations).
#pragma once

// ------------------------------------------------------------------------------------------
// K4 kernel.  LATTICE = false: the tile's pairs come from the list the binning passes K1-K3 wrote.
// LATTICE = true (fused lattice path): the tile enumerates its candidate tets itself.  From K0's slabs each of the
// first three warps finds, for one axis, the first and last cell whose vertex planes reach the tile's sample
// centres: every tet that has a sample in the tile lies in that index box (a superset).  The box's cells are dealt
// to the warps in chunks of 32; a lane whose keep bit is set gathers its tet and takes the exact local box
// (local_box, the one setup_pair uses): only the tets that really reach the tile enter the warp's queue (ballot
// compaction), 32 of which are set up per batch on dense lanes.  No K1/K2/K3, no range array, no pair list; the
// price is the box test of the candidates in the rim of the index box.
// ------------------------------------------------------------------------------------------
template <int NT, int MINB, bool SPARSE, bool LATTICE>
__global__ void __launch_bounds__(NT, MINB) k4_flat(const __grid_constant__ Params p, const u32* __restrict__ offsets,
                                                    const u32* __restrict__ list, u32* __restrict__ bits,
                                                    u32* __restrict__ hdr, const __grid_constant__ SparseOut so,
                                                    const int* __restrict__ slab) {
    __shared__ u32 img[32 * (32 + IMG_SKEW)];
    __shared__ __align__(16) int rec[REC_WORDS(NT)];
    __shared__ int s_incl[NT];  // inclusive scan of the pairs' row counts inside each warp's 32 records
    __shared__ int s_wtot[NT / 32];
    __shared__ u32 s_large;
    __shared__ u32 s_wq[LATTICE ? NT / 32 : 1][LATTICE ? 64 : 1];  // per-warp queue of kept candidates: v0 << 3 | q
    __shared__ int s_rng[LATTICE ? 6 : 1];
    __shared__ u32 s_pairs;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    // tile (bx, by, bz) of mesh m: a 3-D grid (x, y, z*batch) when that fits gridDim (no divisions), else 1-D over tiles
    u32 b, bx, by, bz, m;
    if (p.grid3) {
        bx = blockIdx.x; by = blockIdx.y;
        m = (p.batch == 1) ? 0u : blockIdx.z / (u32)p.nbz;
        bz = blockIdx.z - m * (u32)p.nbz;
        b = ((m * p.nbz + bz) * p.nby + by) * p.nbx + bx;
    } else {
        b = blockIdx.x;
        bx = b % p.nbx;
        u32 rest = b / p.nbx;
        by = rest % p.nby;
        rest /= p.nby;
        bz = rest % p.nbz;
        m = rest / p.nbz;
    }
    const int TY = 1 << p.ty_log, TZ = 1 << p.tz_log;
    TileGeo g;
    g.X0 = bx << 5; g.Y0 = by << p.ty_log; g.Z0 = bz << p.tz_log;
    g.ymax = min(TY, p.ny - g.Y0) - 1;
    g.zmax = min(TZ, p.nz - g.Z0) - 1;
    g.p0x = p.hx * g.X0 + (p.hx >> 1); g.p0y = p.hy * g.Y0 + (p.hy >> 1); g.p0z = p.hz * g.Z0 + (p.hz >> 1);
    g.img_stride = TY + IMG_SKEW;
    g.img_saddr = (u32)__cvta_generic_to_shared(img);
    const u32 rec_saddr = (u32)__cvta_generic_to_shared(rec);
    const int img_stride = g.img_stride;
    const int img_words = img_stride << p.tz_log;
    u32 base = 0, end = 0;
    // LATTICE: candidate index box [ci0, ci0+ni) x [cj0, cj0+nj) x [ck0, ck0+nk), ncand = 6 * cells
    int ci0 = 0, cj0 = 0, ck0 = 0, nj = 1, nk = 1, wq_n = 0;
    u32 ncell = 0, chunk = warp, my_pairs = 0;
    int grp = 0;  // next group of the current chunk (fill stage)
    const u32 cell_base = m * (u32)p.lcx, vert_base = m * (u32)(p.lcx + 1);  // (32-bit: cells and vertices are below 2^31)
    // LATTICE: lane = (cell lane_c of the chunk's five, tet lane_q of the cell's six); tet q walks from the cell's low
    // corner along the axes of the q-th permutation of (x,y,z), lexicographic: xyz xzy yxz yzx zxy zyx (lattice_ids)
    const int lane_c = lane / 6, lane_q = lane - 6 * lane_c;
    const int lat_sy = p.lcz + 1, lat_sx = (p.lcy + 1) * (p.lcz + 1), a123 = lat_sx + lat_sy + 1;
    const int lane_a1 = (lane_q < 2) ? lat_sx : (lane_q < 4) ? lat_sy : 1;
    const int lane_a12 = a123 - ((lane_q == 3 || lane_q == 5) ? lat_sx : (lane_q == 1 || lane_q == 4) ? lat_sy : 1);
    float rnk = 0.f, rnj = 0.f;
    bool small_box = false;
    if (!LATTICE) {
        base = offsets[b];
        end = min(offsets[b + 1], p.cap);
        if (SPARSE && base >= end) {  // no tets: empty tile, nothing else to do
            if (tid == 0) so.table[b] = TILE_EMPTY;
            return;
        }
    } else {
        if (warp < 3) {
            const int c = warp == 0 ? p.lcx : warp == 1 ? p.lcy : p.lcz;  // cells along this warp's axis
            const int* lo = slab + (size_t)m * 2 * (p.lcx + p.lcy + p.lcz + 3) +
                            (warp == 0 ? 0 : warp == 1 ? 2 * (p.lcx + 1) : 2 * (p.lcx + 1) + 2 * (p.lcy + 1));
            const int* hi = lo + c + 1;
            const int E = warp == 0 ? p.ex : warp == 1 ? p.ey : p.ez;
            // the tile's sample centres along this axis: [clo, chi]
            const int clo = warp == 0 ? g.p0x : warp == 1 ? g.p0y : g.p0z;
            const int chi = clo + (warp == 0 ? 31 * p.hx : warp == 1 ? g.ymax * p.hy : g.zmax * p.hz);
            int first = 0x7FFFFFFF, last = -1;
            for (int i0 = 0; i0 < c; i0 += 32) {
                const int i = i0 + lane;
                bool reach = false;
                if (i < c) {  // cell i lies between the vertex planes i and i+1
                    const int cmin = E - max(__ldg(lo + i), __ldg(lo + i + 1)), cmax = max(__ldg(hi + i), __ldg(hi + i + 1));
                    reach = (cmax >= clo) && (cmin <= chi);
                }
                const unsigned bal = __ballot_sync(0xFFFFFFFFu, reach);
                if (bal) {
                    first = min(first, i0 + __ffs(bal) - 1);
                    last = max(last, i0 + 31 - __clz(bal));
                }
            }
            if (lane == 0) { s_rng[2 * warp] = first; s_rng[2 * warp + 1] = last; }
        }
        if (tid == 0) s_pairs = 0;
        __syncthreads();
        ci0 = s_rng[0]; cj0 = s_rng[2]; ck0 = s_rng[4];
        const int ni = max(s_rng[1] - ci0 + 1, 0);
        nj = max(s_rng[3] - cj0 + 1, 0);
        nk = max(s_rng[5] - ck0 + 1, 0);
        ncell = (u32)ni * (u32)nj * (u32)nk;
        small_box = ncell < (1u << 21);
        rnk = 1.0f / (float)max(nk, 1);
        rnj = 1.0f / (float)max(nj, 1);
        if (SPARSE && ncell == 0) {
            if (tid == 0) so.table[b] = TILE_EMPTY;
            return;
        }
    }
    for (int i = tid; i < img_words; i += NT) img[i] = 0;
    if (tid == 0) s_large = 0;
    u32 seen_large = 0;
    for (;;) {
        int n, nr = 0;
        if (!LATTICE) {
            if (base >= end) break;
            __syncthreads();
            n = min((u32)NT, end - base);
            if (tid < n) {
                int* r = rec + rec_off(tid);
                const u32 t = list[base + tid];
                VOX_CHECK((i64)t < p.T && base + tid < p.cap, CK_K4_LIST);
                const int4 id = p.lcx ? lattice_ids(p, t) : __ldg(p.tets + t);
                if (p.pow2) setup_pair<true, false>(p, g, id, r);
                else setup_pair<false, false>(p, g, id, r);
                if (r[6] == 0) atomicAdd(&s_large, 1u);
                nr = r[3];  // >= 1 for every pair: large pairs carry a one-row header that draws nothing
            }
            base += NT;
        } else {
            // fill this warp's queue until it holds a batch's worth.  A chunk is 32 cells of the index box, one per
            // lane: decode the cell, fetch its keep byte (a chunk without kept tets costs just that).  Its candidates
            // are then taken in groups of 5 cells x 6 tets (lane = (lane_c, lane_q), the cell's data by shuffle): a lane
            // whose keep bit is set gathers its tet and takes the exact local box; the tets that reach the tile are
            // appended to the queue.  When the queue is full in mid-chunk the walk stops after group grp and the next
            // batch resumes there (the chunk's decode is simply done again).
            u32* wq = s_wq[warp];
            while (wq_n < 32 && chunk * 32u < ncell) {
                const u32 cell = chunk * 32u + lane;
                u32 kb = 0;
                int v0 = 0;
                if (cell < ncell) {
                    u32 t2, di;
                    if (small_box) {  // exact for cell < 2^21: (cell + 0.5)/nk is at least 0.5/nk away from an integer
                        t2 = (u32)__float2int_rz(((float)cell + 0.5f) * rnk);
                        di = (u32)__float2int_rz(((float)t2 + 0.5f) * rnj);
                    } else {
                        t2 = cell / (u32)nk;
                        di = t2 / (u32)nj;
                    }
                    const u32 i = ci0 + di, j = cj0 + (t2 - di * (u32)nj), k = ck0 + (cell - t2 * (u32)nk);
                    VOX_CHECK(i < (u32)p.lcx && j < (u32)p.lcy && k < (u32)p.lcz, CK_K4_CELL);
                    kb = __ldg(p.keep + (size_t)(((cell_base + i) * p.lcy + j) * p.lcz + k)) & 63u;
                    v0 = (int)(((vert_base + i) * (p.lcy + 1) + j) * (p.lcz + 1) + k);
                }
                const unsigned any = __ballot_sync(0xFFFFFFFFu, kb != 0);
                if (any) {
                    for (; grp < 7; ++grp) {
                        if (((any >> (5 * grp)) & 31u) == 0) continue;  // none of the group's five cells keeps a tet
                        const int src = 5 * grp + lane_c;
                        const u32 kbs = __shfl_sync(0xFFFFFFFFu, kb, src & 31);
                        const int v0s = __shfl_sync(0xFFFFFFFFu, v0, src & 31);
                        bool hit = false;
                        if (lane < 30 && src < 32 && ((kbs >> lane_q) & 1u)) {
                            const Tet q = gather_tet<true>(p, make_int4(v0s, v0s + lane_a1, v0s + lane_a12, v0s + a123));
                            LocalBox B;
                            hit = p.pow2 ? local_box<true>(p, g, q, B) : local_box<false>(p, g, q, B);
                        }
                        const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
                        VOX_CHECK(wq_n + __popc(bal) <= 64, CK_K4_QUEUE);
                        if (hit) wq[wq_n + __popc(bal & ((1u << lane) - 1u))] = ((u32)v0s << 3) | (u32)lane_q;
                        wq_n += __popc(bal);
                        if (wq_n >= 32) { ++grp; break; }
                    }
                } else {
                    grp = 7;
                }
                if (grp >= 7) { grp = 0; chunk += NW; }
            }
            __syncwarp();
            const int take = min(32, wq_n);
            if (!__syncthreads_or(take > 0)) break;  // (also the barrier that frees rec and s_incl)
            n = NT;
            int* r = rec + rec_off(tid);
            bool drawn = false;
            u32 carry = 0;
            if (lane + 32 < wq_n) carry = wq[lane + 32];
            if (lane < take) {
                const u32 e = wq[lane];
                const int v0 = (int)(e >> 3), q = (int)(e & 7u);
                const int a1 = (q < 2) ? lat_sx : (q < 4) ? lat_sy : 1;
                const int a3 = (q == 3 || q == 5) ? lat_sx : (q == 1 || q == 4) ? lat_sy : 1;
                const int4 id = make_int4(v0, v0 + a1, v0 + a123 - a3, v0 + a123);
                drawn = p.pow2 ? setup_pair<true, true>(p, g, id, r) : setup_pair<false, true>(p, g, id, r);
                if (r[6] == 0) atomicAdd(&s_large, 1u);
            } else {
                null_record(r, g.img_saddr);
            }
            nr = r[3];
            my_pairs += __popc(__ballot_sync(0xFFFFFFFFu, drawn));
            __syncwarp();
            if (lane + 32 < wq_n) wq[lane] = carry;  // the rest of the queue moves to the front
            wq_n -= take;
        }
        int incl = nr;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        s_incl[tid] = incl;
        if (lane == 31) s_wtot[warp] = incl;
        __syncthreads();
        // rows of the batch laid end to end: warp segment w covers [cum[w], cum[w+1])
        int cum[NW + 1];
        cum[0] = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) cum[w + 1] = cum[w] + s_wtot[w];
        const int total = cum[NW];
        const int R = (total + NT - 1) / NT;
        const int first = tid * R;
        int cnt = min(R, total - first);
        if (cnt > 0) {
            int w = 0, wb = 0;
#pragma unroll
            for (int k = 1; k < NW; ++k)
                if (first >= cum[k]) { w = k; wb = cum[k]; }
            const int local = first - wb;
            const int* inc = s_incl + w * 32;
            int j = 0;  // smallest j with inc[j] > local
#pragma unroll
            for (int step = 16; step; step >>= 1)
                if (inc[j + step - 1] <= local) j += step;
            int pi = w * 32 + j;
            int rr = local - (j ? inc[j - 1] : 0);
            VOX_CHECK(pi >= 0 && pi < NT && rr >= 0, CK_K4_RECIDX);
            LaneRec L;
            u32 ra = rec_saddr + 4u * (u32)rec_off(pi);
            lane_load(ra, L);
            for (;;) {
                lane_row(L, rr, img_stride, g.img_saddr, g.img_saddr + 4u * (u32)img_words);
                if (--cnt == 0) break;
                if (++rr == L.A.w) {  // next pair (every pair has at least one row)
                    ra += ((++pi & 3) == 0) ? 4u * SREC_W + 16u : 4u * SREC_W;  // rec_off: 16-byte pad after every 4th record
                    VOX_CHECK(pi < NT && ra == rec_saddr + 4u * (u32)rec_off(pi), CK_K4_RECIDX);
                    lane_load(ra, L);
                    rr = 0;
                }
            }
        }
        // large pairs of this batch (rare): one warp per pair, int64 ballot rasteriser
        const u32 nl = s_large;  // cumulative; stable between the barrier above and the next one
        if (nl != seen_large) {
            seen_large = nl;
            for (int i = warp; i < n; i += NW) {
                const int* r = rec + rec_off(i);
                if (r[6] == 0) raster_large_rec(r, img, lane, img_stride);
            }
        }
    }
    if (LATTICE && lane == 0 && my_pairs) atomicAdd(&s_pairs, my_pairs);
    __syncthreads();
    if (tid == 0 && s_large) atomicAdd(hdr + H_LARGE, s_large);
    if (LATTICE && tid == 0 && s_pairs) {  // the statistics K2 leaves in the header on the binned path
        const u32 np = s_pairs, old = atomicAdd(hdr + H_TOTAL, np);
        if (old + np < old) atomicAdd(hdr + H_TOTAL_HI, 1u);
        atomicAdd(hdr + H_NONEMPTY, 1u);
    }
    tile_epilogue<NT, SPARSE>(p, img, img_stride, b, bx, m, g.Y0, g.Z0, bits, hdr, so, tid);
}
