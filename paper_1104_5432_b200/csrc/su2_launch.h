// su2_launch.h — host-side launchers shared by the translation units of libsu2hb.so.
// (Internal to the library; the public boundary is include/su2_heatbath.h.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "su2_device.cuh"

namespace su2 {

// Tiles of one CTA of the tiled heat-bath launch, log2 threads along (hx, y, z, t); 128
// threads each. The first shape whose extents divide the lattice is used, else the
// linear launch (shapes chosen by measurement, profiles/r01b.md).
#ifndef HB_T0
#define HB_T0 4
#define HB_T1 2
#define HB_T2 1
#define HB_T3 0
#endif
constexpr int kNumTiles = 2;
constexpr int kTiles[kNumTiles][4] = {{HB_T0, HB_T1, HB_T2, HB_T3},  // 16 x 4 x 2 x 1 (32 sites along x)
                                      {3, 2, 1, 1}};                  //  8 x 4 x 2 x 2 (16 sites along x)
constexpr int kBlock = 256;                 // block size of every other kernel; part of the
                                            // definition of the fixed-order reductions

// One launch through cudaLaunchKernelEx; `overlap` adds the programmatic-stream-
// serialization attribute (the kernel may start while its predecessor drains).
template <typename... KArgs, typename... Args>
inline void launch_ex(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, bool overlap, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = overlap ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, args...);
}

struct Scratch {
    double* partials;   // [device] block partial sums (plaquette | polyakov | correlator)
    size_t n_partials;  // capacity in doubles
    double* epart;      // [device] fused plaquette partials: 2 sets (su2_run's tail overlap alternates them) of
                        // 3 * heatbath_ctas(g) doubles per replica
    double* field;      // [device] l(x) of the Polyakov kernel, V/Nt doubles
    double* out;        // [device] 2 + kMaxR doubles: plaquette, polyakov, correlator
    int* err;           // [device] sticky error flags (bit 0: KP trial cap hit)
    RunState* state;    // [device] loop state of su2_run: 2 sets of kRunCopies copies
    double* slots;      // [device] step tail: 2 doubles per CTA of the Polyakov kernel (<= V/Nt/64 + 1 CTAs), per replica
    unsigned* ticket;   // [device] step tail: arrival counters (one per replica), zero between steps
    RepParams* reps;    // [device] batch: per-replica 1/beta and seed
};
constexpr int kMaxR = 128;

// Time slab of a lattice split over GPUs: what a sub-step launch needs beyond Geom.
struct SlabCtx {
    uint32_t s_off;          // global site index - local site index (mod 2^32)
    void* peer_lo;           // [device, possibly peer] link buffer of the slab below
    void* peer_hi;           // ... of the slab above
    uint32_t vh_lo, vh_hi;   // links per (p,mu) array of those buffers
    int d_lo, d_hi;          // own link index -> index of its halo copy there
};

// fills g.tile (index into kTiles or -1), g.nb and g.zmagic; nrep = replicas of a batch (grid z = replica x z-t tiles)
void choose_tiling(Geom& g, int nrep = 1, int precision = 64);
size_t partials_needed(const Geom& g);

// each returns the number of kernels it enqueued (0 on launch failure; check cudaGetLastError)
int launch_init(void* links, const Geom& g, int precision, int start, uint64_t seed, cudaStream_t st, int t_shift = 0,
                int nt_glob = 0);
int launch_heatbath_substep(void* links, const Geom& g, int precision, int mu, int parity, double beta,
                            double creutz_below, uint64_t seed, uint32_t sweep, int* err, double* epart,
                            const RunState* state, bool overlap, cudaStream_t st, const RepParams* reps = nullptr,
                            int nrep = 1, const SlabCtx* slab = nullptr);
size_t heatbath_ctas(const Geom& g);
int launch_final_sum(const double* partials, size_t n, double scale, double* dev_dst, cudaStream_t st);
int launch_set_run_state(RunState* state, double inv_beta, double* out, uint32_t sweep, uint32_t index,
                         cudaStream_t st);
// Polyakov partials only (no final sum)
int launch_polyakov_partials(const void* links, const Geom& g, int precision, const Scratch& sc, size_t* n_partials,
                             cudaStream_t st);
int launch_polyakov_step(const void* links, const Geom& g, int precision, const Scratch& sc, const double* epart,
                         size_t n_epart, double scale_plaq, double* dev_dst, RunState* state, bool overlap,
                         cudaStream_t st, int nrep = 1, unsigned advance = 1);
// `scale` = 0: 1 / (number of plaquettes of g); a slab passes 1 / (plaquettes of the whole lattice)
int launch_plaquette(const void* links, const Geom& g, int precision, const Scratch& sc, double* dev_dst,
                     cudaStream_t st, double scale = 0.0);
// slab: continue the ordered product of time links through the interior slices; prev (nullable) = the
// product so far per spatial site, next (nullable) = where to store it, dev_dst (nullable) = mean of 1/2 Tr
int launch_polyakov_chain(const void* links, const Geom& g, int precision, const Scratch& sc, const void* prev,
                          void* next, double* dev_dst, cudaStream_t st);
int launch_polyakov(const void* links, const Geom& g, int precision, const Scratch& sc, double* dev_dst,
                    cudaStream_t st);
int launch_polyakov_correlator(const Geom& g, const Scratch& sc, int rmax, double* dev_dst, cudaStream_t st);
int launch_to_device_layout(const void* canonical, void* links, const Geom& g, int precision, cudaStream_t st);
int launch_to_canonical(const void* links, void* canonical, const Geom& g, int precision, cudaStream_t st);

// no-allocation mean plaquette (su2_measure.cu): partials in a file-scope static __device__ array; returns an SU2_* code
int launch_plaquette_noalloc(const void* links, const Geom& g, int precision, double* dev_dst, cudaStream_t st);
size_t noalloc_max_partials();
// su2_probe.cu: returns an SU2_* code
int run_bandwidth_probe(size_t bytes, int passes, int mode, cudaStream_t st, double* gbs_out, double* us_per_pass_out);

}  // namespace su2
