// sso_ring.cuh -- the contiguous-axis pass of a 2D/3D lattice as an asynchronous ring pipeline (sm_100a).
//
// The last lattice axis is contiguous in memory, so a tile of TL whole lines is one contiguous block.  One
// persistent CTA per SM owns a set of shared-memory buffers.  A tile is fetched by the bulk-copy engine
// (cp.async.bulk, SASS UBLKCP) onto an mbarrier.  G independent groups of GT threads, each with its own
// buffers, take tiles as they become free and, with the tile in registers (16 points per thread) and its
// buffer as the exchange area, apply
//
//   MODE_OPEN   V/2 (natural order)  ->  forward DIF  ->  natural frequency order
//   MODE_MID    inverse DIF  ->  merged potential phase V (permuted order)  ->  forward DIT
//   MODE_CLOSE  inverse DIF  ->  natural order  ->  V/2
//   MODE_CLOSE_OBS  the same, and the observables of the result (norm, autocorrelation with a reference state, <r>,
//               one term of the eigenfunction filter) accumulated before it is stored
//
// (eq. 7, 98 eq. 11; the FFT stages are those of sso_pass.cuh).  As soon as the last exchange of a
// tile has been read, the group's leader claims the next tile of the CTA, refills the buffer and asks L2 for
// that tile's potential-phase lines; the results are stored from registers (512 contiguous bytes per warp
// instruction).  The pass is launched with programmatic dependent launch: its setup overlaps the drain of the
// previous pass of the stream, and it waits (griddepcontrol.wait) before it touches psi.
#pragma once
#include "sso_pass.cuh"

namespace sso {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred P;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P, [%0], %1;\n"
        "@P bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_load(void *smem_dst, const void *gsrc, unsigned bytes, void *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_store(void *gdst, const void *smem_src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// streamed table loads: read once per pass, so keep them out of L1 and first in line for eviction from L2
// (psi of the L2-sized configs then stays resident between passes)
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ double2 ld_table(const double2 *p, uint64_t pol) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_table(const float2 *p, uint64_t pol) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double ld_table(const double *p, uint64_t pol) {
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
// plain streamed table load (read once per pass, shared by the lanes of a k point)
__device__ __forceinline__ double2 ld_table(const double2 *p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void prefetch_l2_bulk_hint(const void *p, unsigned bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(p), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void prefetch_l2_bulk_plain(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// Tile buffers of a persistent CTA: NB shared-memory buffers shared by G compute groups (NB >= G).  The CTA's tiles
// 0 .. nloc-1 are loaded in that order, each into whichever buffer is free: the first NB go to buffers 0 .. NB-1,
// and every time a group has emptied a buffer its leader claims the next unloaded tile for it.  Groups consume the
// tiles in the same order: a leader draws a ticket s (= the s-th tile of the CTA) from a counter, and the group looks
// for the buffer that holds tile s (every buffer carries the number of its tile and the parity of its fill, written
// when the fill is issued) and waits for it there.  With NB > G the spare buffers hold tiles that are loading or
// ready while all groups compute, so a group that finishes finds its next tile already on chip; with NB = G a group
// simply gets back the buffer it refilled.
// A waiter cannot be a fill ahead of its barrier's phase: a buffer is tagged with tile s only when that fill is issued,
// i.e. after the buffer's previous fill has been consumed, and it keeps the tag until the group that drew ticket s has
// worked on it -- however long that group takes.  (A fixed ticket -> buffer map does not have that property: a group
// can lap a slow one and wait on a buffer whose previous fill has not even landed, and the parity of its wait then
// matches a phase that is two fills old.  tests/test_tile_pool_protocol.py is a model of both.)
struct TileRing {
    unsigned long long *bar;  // [NB] "tile landed" barriers
    volatile int *tag;        // [NB] tag[b] = (tile + 1) << 1 | parity of the fill that brings it, 0: never filled
    volatile int *fills;      // [NB] fills issued into each buffer so far
    int *next;                // next unloaded tile of the CTA
    int *ticket;              // next ticket
    volatile int *mail;       // [G] the ticket each group works on next
    int NB, G;
    __device__ TileRing(void *base, int nb, int g) : NB(nb), G(g) {
        bar = reinterpret_cast<unsigned long long *>(base);
        tag = reinterpret_cast<volatile int *>(bar + nb);
        fills = tag + nb;
        next = const_cast<int *>(fills) + nb;
        ticket = next + 1;
        mail = ticket + 1;
    }
    static __host__ __device__ size_t bytes(int nb, int g) { return (size_t)nb * 16 + 8 + (size_t)g * 4; }
    __device__ void *full(int b) const { return bar + b; }
    // once per CTA, by thread 0, before the __syncthreads that precedes the first fill
    __device__ void init() const {
        if (threadIdx.x == 0) {
            for (int b = 0; b < NB; ++b) {
                mbar_init(bar + b, 1);
                fills[b] = 0;
                tag[b] = 0;
            }
            *next = NB;  // tiles 0 .. NB-1 go to buffers 0 .. NB-1
            *ticket = 0;
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    // by the thread that issues the load of tile s into buffer b (one issuer per buffer at a time): tag the buffer;
    // the caller arms the barrier and starts the copy
    __device__ void publish(int s, int b) const {
        const int f = fills[b];
        fills[b] = f + 1;
        tag[b] = ((s + 1) << 1) | (f & 1);
    }
    // group leader: draw the group's next ticket; the group barrier that follows publishes it
    __device__ void draw(int grp) const { mail[grp] = atomicAdd(ticket, 1); }
    __device__ int drawn(int grp) const { return mail[grp]; }
    // blocks until tile s (< nloc) has landed; returns its buffer.  The poll for a fill that has not been issued yet
    // is bounded: a tile of this CTA is issued within a pass (milliseconds), so 2^27 polls of >= 64 ns each (> 8 s)
    // mean the protocol is broken, and the kernel traps (the launch then fails with an error) instead of hanging.
    __device__ int wait(int s) const {
        for (unsigned polls = 0;; ++polls) {
            for (int b = 0; b < NB; ++b) {
                const int v = tag[b];
                if ((v >> 1) == s + 1) {
                    mbar_wait(bar + b, (unsigned)(v & 1));
                    return b;
                }
            }
            if (polls >> 27) __trap();
            __nanosleep(64);  // the load of tile s has not been issued yet
        }
    }
    __device__ int claim() const { return atomicAdd(next, 1); }
};

template <typename T, int N, int MODE, int SIGN, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) ring_kernel(const RingArgs a) {
    using C = typename CxOf<T>::type;
    constexpr int U = N / 16;
    constexpr int LAST = Sched<N>::M - 1;
    constexpr int TWN = Sched<N>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;
    constexpr bool EARLY = MODE == MODE_MID && (sizeof(T) == 4 || MAXT == 384);
    constexpr bool OBS = MODE == MODE_CLOSE_OBS;
    constexpr bool TWG = twiddles_in_global<C, N>();  // the longest lines read their twiddles from global memory
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const C *stw = TWG ? reinterpret_cast<const C *>(a.tw) : reinterpret_cast<const C *>(smem_raw);
    C *bufs = reinterpret_cast<C *>(smem_raw) + (TWG ? 0 : TWP);
    TileRing ring(bufs + (size_t)a.NB * a.bufstride, a.NB, a.G);

    const int TL = a.TL, GT = a.GT, G = a.G, NB = a.NB;
    const int grp = threadIdx.x / GT;
    const int tid = threadIdx.x - grp * GT;
    // lanes of a warp hold consecutive u (and whole lines when U < 32): stage exchanges that stay inside 32
    // consecutive u need no group barrier
    const int gb = (G > 1 ? ((grp + 1) | (GT << 8)) : 0) | ((U >= 32 || 32 % U == 0) ? GB_LANES_ARE_U : 0);
    const int u = tid % U;
    const int t = tid / U;
    const unsigned tile_bytes = (unsigned)(TL * N * sizeof(C));
    const int nloc = a.ntiles > (int)blockIdx.x ? (a.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const uint64_t pol = policy_evict_first();
    const size_t vesz = a.vrep == VREP_TABLE ? sizeof(C) : sizeof(double);
    C *gpsi = reinterpret_cast<C *>(a.psi);

    // issue the load of local tile k into its ring buffer, and ask L2 for that tile's potential-phase lines
    // tile -> first element of psi and first potential-table line (component fastest)
    auto tile_elem = [&](long long tile, long long *table_line) {
        const long long comp = tile & (a.ncomp - 1), lb = tile >> a.ncomp_shift;  // ncomp is 1, 2 or 4
        *table_line = lb * TL;
        return (comp * a.lines_per_comp + lb * TL) * (long long)N;
    };
    // CTA-local tile k -> global tile.  rev: highest addresses first, so that this pass starts on what the previous
    // pass of the stream (which ended there) left in L2 and ends on the lowest addresses, where the next one starts
    auto tile_of = [&](int k) -> long long {
        const long long tl = (long long)blockIdx.x + (long long)k * gridDim.x;
        return a.rev ? (long long)a.ntiles - 1 - tl : tl;
    };
    auto issue = [&](int k, int b) {
        const long long tile = tile_of(k);
        long long l0;
        const long long e0 = tile_elem(tile, &l0);
        mbar_expect_tx(ring.full(b), tile_bytes);
        bulk_load(bufs + (size_t)b * a.bufstride, gpsi + e0, tile_bytes, ring.full(b));
        if (a.vtab && (tile & (a.ncomp - 1)) == 0)  // one request per table block
            prefetch_l2_bulk_plain(reinterpret_cast<const char *>(a.vtab) + (size_t)l0 * N * vesz, (unsigned)(TL * N * vesz));
    };

    // let the next pass of the stream start its own setup as SMs free up
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    ring.init();
    if constexpr (!TWG) {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        C *dst = reinterpret_cast<C *>(smem_raw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) dst[i] = gtw[i];
    }
    __syncthreads();
    // everything above touched only plan-owned tables; psi is valid once the previous pass has completed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // hand a buffer its next tile, if there is one left
    auto refill = [&](int kn, int b) {
        if (kn < nloc) {
            ring.publish(kn, b);
            issue(kn, b);
        }
    };
    if (tid == 0) {
        for (int b = grp; b < NB; b += G) refill(b, b);  // the first NB tiles, loaded by the groups' leaders
        ring.draw(grp);
    }
    gsync(gb);  // publishes the group's first ticket

    // MODE_CLOSE_OBS: per-thread sums over all the tiles this thread meets
    [[maybe_unused]] double ob[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    [[maybe_unused]] double fwr = 0.0, fwi = 0.0;
    if constexpr (OBS) {
        if (a.facc) {
            sincos(a.fw_E * a.fw_t, &fwi, &fwr);
            const double wdw = (1.0 - cospi(2.0 * a.fw_t / a.fw_T)) * a.fw_dts;
            fwr *= wdw;
            fwi *= wdw;
        }
    }

    for (;;) {
        const int k = ring.drawn(grp);  // the group's next tile, in the CTA's loading order
        if (k >= nloc) break;
        const int b = ring.wait(k);
        C *buf = bufs + (size_t)b * a.bufstride;
        C *dense = buf + t * N + u;          // bulk-copy layout: [TL][N]
        C *sl = buf + t * a.pitch;           // exchange layout: padded lines
        const long long tile = tile_of(k);
        long long l0_;
        const long long e0_ = tile_elem(tile, &l0_);
        const int lic = (int)l0_ + t;  // line within the component = table line
        const size_t vbase = (size_t)lic * N + u;

        // pointwise factor of this pass for register q (table slot q U + u of line lic)
        // with registers to spare (complex64, or the 384-thread build) the merged-phase line is requested before
        // the tile is even waited for, so that its latency hides behind the first transform
        [[maybe_unused]] C hh[EARLY ? 16 : 1];
        if constexpr (EARLY) {
            if (a.vrep == VREP_TABLE) {
                const C *vt = reinterpret_cast<const C *>(a.vtab) + vbase;
#pragma unroll
                for (int q = 0; q < 16; ++q) hh[q] = ld_table(vt + q * U, pol);
            }
        }
        auto phase = [&](C (&x)[16]) {
            C s = mk<C>((T)1, (T)0);
            bool has_s = false;
            if (a.eoA) {
                s = reinterpret_cast<const C *>(a.eoA)[lic >> a.rest1_shift];
                has_s = true;
            }
            if (a.eoB) {
                const C sb = reinterpret_cast<const C *>(a.eoB)[lic & (a.rest1 - 1)];
                s = has_s ? cmul(s, sb) : sb;
                has_s = true;
            }
            if (a.vrep == VREP_TABLE) {
                const C *vt = reinterpret_cast<const C *>(a.vtab) + vbase;
                if constexpr (EARLY) {
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        C f = hh[q];
                        if (a.eline) f = cmul(f, reinterpret_cast<const C *>(a.eline)[q * U + u]);
                        if (has_s) f = cmul(f, s);
                        x[q] = cmul(x[q], f);
                    }
                } else {
                    C h[8];
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
#pragma unroll
                        for (int q = 0; q < 8; ++q) h[q] = ld_table(vt + (half * 8 + q) * U, pol);
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            C f = h[q];
                            if (a.eline) f = cmul(f, reinterpret_cast<const C *>(a.eline)[(half * 8 + q) * U + u]);
                            if (has_s) f = cmul(f, s);
                            x[half * 8 + q] = cmul(x[half * 8 + q], f);
                        }
                    }
                }
            } else {
                const double *vt = reinterpret_cast<const double *>(a.vtab) + vbase;
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    C f = expi_small<T>(ld_table(vt + q * U, pol));
                    if (a.eline) f = cmul(f, reinterpret_cast<const C *>(a.eline)[q * U + u]);
                    if (has_s) f = cmul(f, s);
                    x[q] = cmul(x[q], f);
                }
            }
        };
        C x[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = dense[q * U];
        gsync(gb);  // the exchange layout overlaps the bulk-copy layout of other warps' lines

        if constexpr (MODE == MODE_OPEN) phase(x);
        DifChain<T, N, 0, SIGN>::run(x, u, stw, sl, gb);
        if constexpr (MODE == MODE_MID) {
            phase(x);
            DitChain<T, N, LAST, -SIGN>::run(x, u, stw, sl, gb);
        } else {
            // registers hold frequency revB[u] + U q at network position 16 u + q: scatter to natural order
            C *wa = sl + padp(a.revB[u]);
            const C *rb = sl + padp(u);
            gsync(gb);
#pragma unroll
            for (int q = 0; q < 16; ++q) wa[lin_delta(q, U)] = x[q];
            gsync(gb);
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = rb[lin_delta(q, U)];
            if constexpr (MODE == MODE_CLOSE || OBS) phase(x);
        }

        if constexpr (OBS) {
            // x is psi(t) in natural order: register q <-> position u + q U of line lic of component tile mod ncomp
            const size_t e1 = (size_t)e0_ + (size_t)t * N + u;
            double dsum = 0.0, dline = 0.0;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const double d = (double)x[q].x * (double)x[q].x + (double)x[q].y * (double)x[q].y;
                dsum += d;
                dline += d * (double)(u + q * U - a.obs_half[2]);
            }
            ob[0] += dsum;
            if (a.obs_axL >= 0) ob[3 + a.obs_axL] += dline * a.obs_dx[2];
            if (a.obs_axA >= 0) ob[3 + a.obs_axA] += dsum * (double)((lic >> a.rest1_shift) - a.obs_half[0]) * a.obs_dx[0];
            if (a.obs_axB >= 0) ob[3 + a.obs_axB] += dsum * (double)((lic & (a.rest1 - 1)) - a.obs_half[1]) * a.obs_dx[1];
            if (a.ref) {
                const C *gr = reinterpret_cast<const C *>(a.ref) + e1;
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const C r = ld_stream(gr + q * U);
                    ob[1] += (double)r.x * (double)x[q].x + (double)r.y * (double)x[q].y;
                    ob[2] += (double)r.x * (double)x[q].y - (double)r.y * (double)x[q].x;
                }
            }
            if (a.facc) {
                double2 *ga = reinterpret_cast<double2 *>(a.facc) + e1;
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    double2 v = ga[q * U];
                    v.x += fwr * (double)x[q].x - fwi * (double)x[q].y;
                    v.y += fwr * (double)x[q].y + fwi * (double)x[q].x;
                    ga[q * U] = v;
                }
            }
        }

        // the buffer was written with ordinary (generic-proxy) stores and is refilled by the bulk-copy engine (async
        // proxy): every thread orders its accesses before the refill, then the group meets
        fence_async_smem();
        if (tid == 0) ring.draw(grp);  // the group's next ticket, published by the barrier
        gsync(gb);  // every thread of the group is done with the buffer: it can take its next tile right away
        if (tid == 0) refill(ring.claim(), b);
        // results go straight from registers to global memory (512 contiguous bytes per warp instruction):
        // no second trip through shared memory and nothing to wait for before the buffer is refilled
        {
            C *gout = gpsi + e0_ + (size_t)t * N + u;
#pragma unroll
            for (int q = 0; q < 16; ++q) st_stream(gout + q * U, x[q]);
        }
    }
    if constexpr (OBS) {
        // CTA sums by shared-memory atomics, one row of partial sums per CTA (a final kernel adds
        // the rows in a fixed order; which tiles a warp met depends on the tile pool, so the last bits may differ from run to run)
        double *cta = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(bufs + (size_t)a.NB * a.bufstride) + 448);
        __syncthreads();  // every group has left the tile loop
        if (threadIdx.x == 0)  // (a CTA of a tiny lattice may have fewer than six threads)
            for (int v = 0; v < 6; ++v) cta[v] = 0.0;
        __syncthreads();
        // (a CTA of a tiny lattice may hold a partial warp, so no full-mask shuffles here: once per launch, the cost is nil)
#pragma unroll
        for (int v = 0; v < 6; ++v) atomicAdd(&cta[v], ob[v]);
        __syncthreads();
        if (threadIdx.x == 0)
            for (int v = 0; v < 6; ++v) a.obs_partial[(size_t)v * gridDim.x + blockIdx.x] = cta[v];
    }
}

template <typename T, int N, int MODE, int SIGN, int MAXT>
cudaError_t launch_ring(const RingArgs &a, unsigned threads, size_t smem, unsigned grid, cudaStream_t st);

}  // namespace sso
