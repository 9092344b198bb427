// kernels_bin.cuh -- part of vox.cu (included there, once): the binning passes K1 (count), K2 (scan), K3 (scatter).
#pragma once

// ------------------------------------------------------------------------------------------
// K1: per-tet voxel bbox -> tile range, cull, histogram
// ------------------------------------------------------------------------------------------
#define RANGE_CULLED 0xFFFFFFFFu

__global__ void __launch_bounds__(256) k1_count(Params p, uint2* __restrict__ range, u32* __restrict__ counts,
                                                u32* __restrict__ hdr, u32* __restrict__ big) {
    i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = false, handed = false;
    uint2 r = make_uint2(RANGE_CULLED, 0u);
    int m = 0;
    int b0x = 0, b1x = -1, b0y = 0, b1y = -1, b0z = 0, b1z = -1;
    const bool present = (t < p.T) && (!p.lcx || ((__ldg(p.keep + (u32)t / 6u) >> (int)((u32)t % 6u)) & 1));
    // (lattice input: a tet its cell does not keep gets no range entry -- K3 looks at the keep bit first)
    if (present) {
        Tet q = load_tet(p, t);
        int x0, x1, y0, y1, z0, z1;
        axis_range(q.ax, q.bx, q.cx, q.dx, p.hx, p.qx, p.nx, x0, x1);
        axis_range(q.ay, q.by, q.cy, q.dy, p.hy, p.qy, p.ny, y0, y1);
        axis_range(q.az, q.bz, q.cz, q.dz, p.hz, p.qz, p.nz, z0, z1);
        live = (x0 <= x1) && (y0 <= y1) && (z0 <= z1) && (six_volume(q) != 0);
        if (live) {
            b0x = x0 >> 5; b1x = x1 >> 5;
            b0y = y0 >> p.ty_log; b1y = y1 >> p.ty_log;
            b0z = z0 >> p.tz_log; b1z = z1 >> p.tz_log;
            r.x = (u32)b0x | ((u32)b0y << 10) | ((u32)b0z << 20);
            r.y = (u32)b1x | ((u32)b1y << 10) | ((u32)b1z << 20);
            m = mesh_of(p, t);
            if ((b1x - b0x + 1) * (b1y - b0y + 1) * (b1z - b0z + 1) > BIG_TILES) {  // oversized: hand over to K2
                const u32 slot = atomicAdd(hdr + H_NBIG, 1u);
                if (slot < (u32)BIG_CAP) {
                    big[slot] = (u32)t;
                    r.x |= RANGE_BIG;
                    handed = true;
                }
            }
        }
        range[t] = r;
    }
    unsigned dead = __ballot_sync(0xFFFFFFFFu, present && !live);
    if ((threadIdx.x & 31) == 0 && dead) atomicAdd(hdr + H_CULLED, __popc(dead));
    // warp-aggregated histogram: in step k every live lane names the k-th tile of its range; lanes
    // naming the same tile (neighbouring tets mostly do) are merged into one atomic
    live = live && !handed;
    int cx = b0x, cy = b0y, cz = b0z;
    const u32 lt = (1u << (threadIdx.x & 31)) - 1u;
    for (;;) {
        const unsigned act = __ballot_sync(0xFFFFFFFFu, live);
        if (!act) break;
        if (live) {
            const u32 b = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(b < p.NB, CK_K1_TILE);
            const unsigned peers = __match_any_sync(act, b);
            // (the group's lowest lane adds for all of it; "no peer below me" is a LOP on the alu pipe where
            //  lane == __ffs(peers) - 1 cost a BREV + FLO on the quarter-rate XU pipe)
            if ((peers & lt) == 0) atomicAdd(counts + b, (u32)__popc(peers));
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// K2: exclusive scan of counts[0..NB) (single CTA, 4096 counters per pass; NB is at most a few 10^5)
// counts[b] <- offset, counts[NB] <- total, cursor[b] <- offset
// ------------------------------------------------------------------------------------------
// tile b of the idx-th tile of a packed range
__device__ __forceinline__ u32 range_tile(const Params& p, uint2 r, int m, u32 idx) {
    const u32 b0x = r.x & 1023, b0y = (r.x >> 10) & 1023, b0z = (r.x >> 20) & 1023;
    const u32 wx = (r.y & 1023) - b0x + 1, wy = ((r.y >> 10) & 1023) - b0y + 1;
    const u32 dx = idx % wx, rest = idx / wx;
    const u32 dy = rest % wy, dz = rest / wy;
    return ((((u32)m * p.nbz + b0z + dz) * p.nby + b0y + dy) * p.nbx) + b0x + dx;
}
__device__ __forceinline__ u32 range_tiles(uint2 r) {
    const u32 wx = (r.y & 1023) - (r.x & 1023) + 1, wy = ((r.y >> 10) & 1023) - ((r.x >> 10) & 1023) + 1;
    const u32 wz = ((r.y >> 20) & 1023) - ((r.x >> 20) & 1023) + 1;
    return wx * wy * wz;
}

__global__ void __launch_bounds__(1024) k2_scan(Params p, const uint2* __restrict__ range, const u32* __restrict__ big,
                                                u32* __restrict__ list, u32* __restrict__ counts,
                                                u32* __restrict__ cursor, u32* __restrict__ hdr, int scatter_big) {
    const u32 NB = p.NB;
    // oversized tets (K1 listed them): the whole CTA counts their tiles, 1024 at a time
    const u32 nbig = min(hdr[H_NBIG], (u32)BIG_CAP);
    for (u32 e = 0; e < nbig; ++e) {
        const u32 t = big[e];
        const uint2 r = range[t];
        const int m = mesh_of(p, t);
        const u32 n = range_tiles(r);
        for (u32 idx = threadIdx.x; idx < n; idx += 1024u) {
            VOX_CHECK(range_tile(p, r, m, idx) < p.NB, CK_K2_TILE);
            atomicAdd(counts + range_tile(p, r, m, idx), 1u);
        }
    }
    if (nbig) {
        __threadfence();
        __syncthreads();
    }
    // chunks of 4096 counters: one coalesced uint4 per thread, warp shuffle scan, 32 warp partials
    // scanned by warp 0, running carry in 64 bits (a total above 2^32 raises the overflow flag)
    __shared__ u64 s_warp[32];
    __shared__ u64 s_carry;
    __shared__ u32 s_ne[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool vec_ok = ((size_t)counts & 15) == 0 && ((size_t)cursor & 15) == 0;
    if (tid == 0) s_carry = 0;
    u32 ne = 0;
    auto load4 = [&](u32 i) {
        uint4 c = make_uint4(0u, 0u, 0u, 0u);
        if (i + 3 < NB && vec_ok) c = __ldcg(reinterpret_cast<const uint4*>(counts + i));
        else {
            if (i < NB) c.x = __ldcg(counts + i);
            if (i + 1 < NB) c.y = __ldcg(counts + i + 1);
            if (i + 2 < NB) c.z = __ldcg(counts + i + 2);
            if (i + 3 < NB) c.w = __ldcg(counts + i + 3);
        }
        return c;
    };
    uint4 nxt = load4((u32)tid * 4u);
    for (u32 base = 0; base < NB; base += 4096u) {
        const u32 i = base + (u32)tid * 4u;
        const uint4 c = nxt;
        if (base + 4096u < NB) nxt = load4(i + 4096u);  // prefetch the next chunk
        ne += (c.x != 0) + (c.y != 0) + (c.z != 0) + (c.w != 0);
        const u64 mine = (u64)c.x + c.y + c.z + c.w;
        u64 incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        __syncthreads();  // s_warp / s_carry of the previous chunk are consumed
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const u64 w = s_warp[lane];
            u64 wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u64 v = __shfl_up_sync(0xFFFFFFFFu, wi, o);
                if (lane >= o) wi += v;
            }
            const u64 carry = s_carry;
            s_warp[lane] = carry + wi - w;  // exclusive offset of each warp, carry included
            __syncwarp();
            if (lane == 31) s_carry = carry + wi;
        }
        __syncthreads();
        const u64 run = s_warp[warp] + incl - mine;
        uint4 o4;
        o4.x = (u32)run;
        o4.y = (u32)(run + c.x);
        o4.z = (u32)(run + c.x + c.y);
        o4.w = (u32)(run + c.x + c.y + c.z);
        if (i + 3 < NB && vec_ok) {
            *reinterpret_cast<uint4*>(counts + i) = o4;
            *reinterpret_cast<uint4*>(cursor + i) = o4;
        } else {
            if (i < NB) { counts[i] = o4.x; cursor[i] = o4.x; }
            if (i + 1 < NB) { counts[i + 1] = o4.y; cursor[i + 1] = o4.y; }
            if (i + 2 < NB) { counts[i + 2] = o4.z; cursor[i + 2] = o4.z; }
            if (i + 3 < NB) { counts[i + 3] = o4.w; cursor[i + 3] = o4.w; }
        }
    }
    for (int o = 16; o; o >>= 1) ne += __shfl_xor_sync(0xFFFFFFFFu, ne, o);
    if (lane == 0) s_ne[warp] = ne;
    __syncthreads();
    if (tid == 0) {
        const u64 total = s_carry;
        counts[NB] = (u32)min(total, (u64)0xFFFFFFFFu);
        hdr[H_TOTAL] = (u32)total;
        hdr[H_TOTAL_HI] = (u32)(total >> 32);
        if (total > 0xFFFFFFFFull) hdr[H_OVERFLOW] = 1;
        u32 s = 0;
        for (int k = 0; k < 32; ++k) s += s_ne[k];
        hdr[H_NONEMPTY] = s;
    }
    if (nbig && scatter_big) {  // scatter the oversized tets (K3 appends the others to the same cursors afterwards)
        __threadfence();
        __syncthreads();
        for (u32 e = 0; e < nbig; ++e) {
            const u32 t = big[e];
            const uint2 r = range[t];
            const int m = mesh_of(p, t);
            const u32 n = range_tiles(r);
            for (u32 idx = threadIdx.x; idx < n; idx += 1024u) {
                const u32 pos = atomicAdd(cursor + range_tile(p, r, m, idx), 1u);
                if (pos < p.cap) list[pos] = t;
                else hdr[H_OVERFLOW] = 1;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// K3: scatter tet ids into the per-tile lists
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k3_scatter(Params p, const uint2* __restrict__ range, u32* __restrict__ cursor,
                                                  u32* __restrict__ list, u32* __restrict__ hdr) {
    i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = false;
    int b0x = 0, b0y = 0, b1x = 0, b1y = 0, b1z = 0, cx = 0, cy = 0, cz = 0, m = 0;
    if (t < p.T && (!p.lcx || ((__ldg(p.keep + (u32)t / 6u) >> (int)((u32)t % 6u)) & 1))) {
        const uint2 r = range[t];
        if (r.x != RANGE_CULLED && !(r.x & RANGE_BIG)) {  // (oversized tets were scattered by K2)
            live = true;
            b0x = r.x & 1023; b0y = (r.x >> 10) & 1023; cz = (r.x >> 20) & 1023;
            b1x = r.y & 1023; b1y = (r.y >> 10) & 1023; b1z = (r.y >> 20) & 1023;
            cx = b0x; cy = b0y;
            m = mesh_of(p, t);
        }
    }
    // (tried, round 2: one atomic per (tet, tile) with up to 8 in flight per thread instead of the lockstep aggregation --
    //  2-3.5x slower, 0.15 against 0.072 ms on cfg4, 0.32 against 0.092 on the 10^7-tet mesh: the cursors of a tile are hot
    //  addresses and the number of atomics, not their latency, is what binds)
    // warp-aggregated cursor bump (same stepping as K1): one atomic per distinct tile per step, the lanes of a group
    // take consecutive slots (order inside a tile list is irrelevant: OR).  TWO steps per trip: the kernel is bound by
    // the round trip of the returning atomics, and most tets touch one or two tiles, so the atomics of a lane's next
    // tile are put in flight together with those of its current one.
    const int lane = threadIdx.x & 31;
    const u32 lt = (1u << lane) - 1u;
    for (;;) {
        const unsigned actA = __ballot_sync(0xFFFFFFFFu, live);
        if (!actA) break;
        u32 bA = 0, bB = 0;
        unsigned peersA = 0, peersB = 0;
        bool liveB = false;
        if (live) {
            bA = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(bA < p.NB, CK_K3_TILE);
            peersA = __match_any_sync(actA, bA);
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
            liveB = live;
        }
        const unsigned actB = __ballot_sync(0xFFFFFFFFu, liveB);
        if (liveB) {
            bB = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(bB < p.NB, CK_K3_TILE);
            peersB = __match_any_sync(actB, bB);
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
        }
        // both groups' atomics in flight before either result is used
        u32 baseA = 0, baseB = 0;
        if (peersA && (peersA & lt) == 0) baseA = atomicAdd(cursor + bA, (u32)__popc(peersA));
        if (peersB && (peersB & lt) == 0) baseB = atomicAdd(cursor + bB, (u32)__popc(peersB));
        if (peersA) {
            baseA = __shfl_sync(peersA, baseA, __ffs(peersA) - 1);
            const u32 pos = baseA + (u32)__popc(peersA & lt);
            if (pos < p.cap) list[pos] = (u32)t;
            else hdr[H_OVERFLOW] = 1;
        }
        if (peersB) {
            baseB = __shfl_sync(peersB, baseB, __ffs(peersB) - 1);
            const u32 pos = baseB + (u32)__popc(peersB & lt);
            if (pos < p.cap) list[pos] = (u32)t;
            else hdr[H_OVERFLOW] = 1;
        }
    }
}
