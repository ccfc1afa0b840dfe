/* mcrt_dev.h -- the laboratory side of libmcrt.so: tuning knobs (none of them changes a result:
 * tallies are integers and every package owns its Philox stream), measurement tools and the test
 * hooks the parity tests use.  Not part of the stable boundary (mcrt.h); names and meanings may
 * change between versions.  Same rules as mcrt.h: plain pointers, mcrt_status, no aborts.
 */
#ifndef MCRT_DEV_H_
#define MCRT_DEV_H_

#include "mcrt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Gather-roofline calibration (BASELINE.json metric "% of gather-BW roofline"; SURVEY.md 8(d)
 * item (iv)): times at least `n_gathers` independent, hash-indexed 4-byte gathers over a
 * zero-filled device array of `footprint_bytes` (4 B .. 16 GiB; allocated and freed inside the
 * call) at full occupancy on the current device and returns gathers per second (and the timed
 * seconds if `seconds` is not NULL).  Host output pointers.  It is the ceiling for a cell walk
 * in which every crossing costs one density gather and nothing else; the transport kernels'
 * crossings per second are reported against it by bench.py. */
mcrt_status mcrt_gather_calibrate(uint64_t footprint_bytes, uint64_t n_gathers, double* gathers_per_s,
                                  double* seconds, void* cuda_stream);

/* ---- tuning and introspection (do not change results) ---------------------------------------
 * Launch shape of the transport kernel: threads per block (multiple of 32, <= 256; 0 keeps the
 * current value) and resident blocks per SM (0 = automatic: 5, or 4 for a single-level grid larger
 * than the L2; more than 1024 resident threads per SM select the 48-register build of the kernel). */
mcrt_status mcrt_set_launch(mcrt_ctx* ctx, int32_t threads_per_block, int32_t blocks_per_sm);
/* A warp leaves the cell-walk loop to process its stopped lanes (escape, refill, scattering,
 * absorption) when fewer than `quorum` of its 32 lanes are still walking (1..32).  0 = automatic
 * (the default): 14 + 2 log2(L / 24) clamped to 8..24, L = the job's crossings per flight so far
 * (long free flights -> keep more lanes walking).  A scheduling knob only: results do not depend
 * on it. */
mcrt_status mcrt_set_walk_quorum(mcrt_ctx* ctx, int32_t quorum);
/* End of a batch.  mode bit 0: when the work queue is empty every warp still holds up to 32 packages (PAPER.md
 * L25: the packages of a batch fly together, and the batch is over when the last one has left); the walk quorum
 * then follows the number of packages the warp still holds (the same share of them as in the steady state)
 * instead of dropping to 1.  mode bit 1: mcrt_run_batch runs the temperature update (the cell's
 * energy "and accordingly its temperature") at the end of the transport launch itself, behind a grid-wide
 * barrier (cooperative launch), instead of in a launch of its own -- not on swept grids, with a PAH declared or
 * for packet-sharded batches.  -1 = automatic (the default: bit 0, and bit 1 on grids of at most 65536 leaf
 * slots, where a second launch costs as much as the whole batch: the 16^3 sphere's 10^4-package batches).
 * Scheduling only: results do not depend on it. */
mcrt_status mcrt_set_tail_mode(mcrt_ctx* ctx, int32_t mode);
/* Region sweeps (single-level grids of at least 256^3 cells in the brick layout, batches of at least 2^20
 * packages): the batch is transported in `sweeps` + 1 passes; in all but the last a package that crosses
 * into another region (256 x 128 x 128 cells by default, 128^3 on a 256^3 grid) is suspended (48 bytes of state) and continues in the next pass,
 * where the waiting packages are handed out region by region, so that the cells the packages in flight
 * visit stay in the L2; the last pass finishes whatever is left.  sweeps: -1 = automatic (the default: 6
 * for batches of at least 2^20 packages), 0 = off, 1..30 (then for any batch size).  rx, ry, rz: region
 * edges in cells (multiples of 8 that divide n_root, 2..4096 regions), 0 0 0 = keep.  Results do not
 * depend on any of it (integer tallies, the state is restored exactly). */
mcrt_status mcrt_set_region_sweeps(mcrt_ctx* ctx, int32_t sweeps, int32_t rx, int32_t ry, int32_t rz);
/* Packages suspended in sweep 0, 1, ... of the LAST swept batch (host array of `cap` entries, at most 32
 * are written; *n_out = number written, 0 if no batch was swept yet). */
mcrt_status mcrt_get_region_sweep_counts(mcrt_ctx* ctx, uint32_t* suspended_out, int32_t cap, int32_t* n_out);
/* Density kept in shared memory (single-level grids): a density array of at most 40 KB is copied
 * into every block's shared memory by one bulk copy (cp.async.bulk) and a crossing reads shared
 * memory instead of the L2 (C0: -10 % per launch).  mode 0 = automatic (the default), 1 = off
 * (always gather from global memory), 2 = automatic, and additionally a larger grid that holds
 * only two distinct densities (a uniform sphere in vacuum) is staged as ONE BIT per cell if the
 * bits fit in 40 KB -- kept for measurement: on the 64^3 sphere it is 3 % slower than global
 * gathers (profiles/r02_summary.md).  Results do not depend on it.  mcrt_density_staging returns
 * what the next batch will use: 0 none, 1 the fp32 array, 2 one bit per cell (-1: NULL). */
mcrt_status mcrt_set_density_staging(mcrt_ctx* ctx, int32_t mode);
int32_t mcrt_density_staging(const mcrt_ctx* ctx);
/* Hand the packages of a batch to the lanes grouped by where they start (a pre-pass evaluates the
 * first decisions of every package's emission and groups the package numbers), so that the
 * packages in flight share a neighbourhood and the L2 serves more of their gathers.  mode 1 =
 * grouped by source, 2 = by source and start direction (8 x 16 bins in (mu, phi) for a point
 * source -- 4 x 8 with more than 16 sources --, face x 2 x 2 tiles for the external field), 0 =
 * off, -1 = automatic (2 when the density array is larger than the L2 or the batch has at least
 * 2^21 packages).  Batches below 65536 packages are never reordered; more than 64 sources fall
 * back to mode 1, more than 2048 to 0.  Integer tallies: results do not depend on it. */
mcrt_status mcrt_set_source_order(mcrt_ctx* ctx, int32_t mode);
/* The re-emission bin of an absorbed package is the first bin whose cumulative emission reaches the
 * package's uniform (Eqn 11.67; R11), found by bisection of a table row.  on != 0
 * (the default): a guide table built with the rows (32 slices of the uniform per row) hands the
 * bisection the few bins of the uniform's slice -- one load instead of its first four or five
 * probes; on = 0: plain bisection of the whole row.  The bin found is the same, bit for bit. */
mcrt_status mcrt_set_cdf_guide(mcrt_ctx* ctx, int32_t on);
/* Device times in ms of the mcrt_run_batch calls made since the previous call of this function
 * (oldest first, at most `cap`), split into the two kernels of a batch (transport, temperature
 * update), from CUDA events recorded on each batch's stream.  Synchronises with those streams.
 * *n_out (host) receives the number written.  Either array may be NULL. */
mcrt_status mcrt_get_batch_times(mcrt_ctx* ctx, float* transport_ms, float* update_ms, int32_t cap,
                                 int32_t* n_out);
/* Copies the built tables (fp32, device -> host) for inspection: opac[n_bins][4] = (kappa_ext *
 * root_size, albedo, g, kappa_abs), lnQ[n_T], cdf[n_T][n_bins].  Any pointer may be NULL. */
mcrt_status mcrt_get_tables(mcrt_ctx* ctx, float* opac, float* lnQ, float* cdf);
/* Number of kernels launched by this library since the context was created. */
int64_t mcrt_kernel_launches(const mcrt_ctx* ctx);
/* Library built with -DMCRT_CHECKS (paper_1201_3588_b200/build.py build_library(checks=True)):
 * number of storage-slot indices the transport kernels found outside the grid's storage since
 * the library was loaded (must stay 0); -1 if the library was built without the checks, -2 on
 * a CUDA error.  Stands in for compute-sanitizer, which the GPU pool does not offer. */
int64_t mcrt_debug_violations(void);
/* Raw Philox4x32-10 blocks computed on the device (test hook for the generator pin):
 * out[4*i..4*i+3] = Philox(key = (key2[0], key2[1]), counter = ctr[4*i..4*i+3]).  Host pointers. */
mcrt_status mcrt_philox_blocks(const uint32_t* key2, const uint32_t* ctr, uint32_t* out, int64_t n);
/* The kernels' maps from a random word to a uniform (test hook for reading R19): u[i] = the fp32
 * uniform ((w >> 9) + 0.5) 2^-23 used for every draw of a flight, ud[i] = the fp64 uniform
 * (w + 0.5) 2^-32 used for the two emission decisions (source, frequency bin), tau[i] = -ln u[i]
 * as the free-flight draw computes it.  Both uniforms lie strictly inside (0,1).  Host pointers. */
mcrt_status mcrt_uniforms(const uint32_t* words, float* u, double* ud, float* tau, int64_t n);

#ifdef __cplusplus
}
#endif
#endif /* MCRT_DEV_H_ */
