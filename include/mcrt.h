/* mcrt.h -- C ABI of the B200-native Monte Carlo dust radiative-transfer hot path: the stable
 * boundary (SURVEY.md 8(b) plus the calls of rows e, f1, f2).  Tuning knobs, measurement tools and
 * test hooks live in mcrt_dev.h.
 *
 * Method: Siebenmorgen, Heymann & Kruegel, "PAH in vectorized three dimensional Monte Carlo
 * dust radiative transfer models", section 2:
 *   PAPER.md L23   space partitioned into cubes, some divided into subcubes (cells); the star
 *                  emits photon packages of constant energy eps at different frequencies; in
 *                  each cell on its flight path a package may be absorbed or scattered with a
 *                  probability given by the extinction optical depth along the path in the cell;
 *                  scattering changes the direction by the phase function; absorption raises the
 *                  cell energy by eps (and so its temperature) and a new package of the same
 *                  energy is emitted isotropically from the spot at a new frequency.
 *   PAPER.md L25-27  many packages are followed simultaneously; the new frequency is drawn at
 *                  the cell temperature BEFORE absorption without the Bjorkman-Wood correction
 *                  (Eqn 11.67 instead of 11.65 of Kruegel 2006): dP/dnu ~ kappa_nu B_nu(T).
 * The call names are the ones BASELINE.json north_star fixes; everything below the names is this
 * build's reading (readings R1..R33).
 *
 * General rules
 *  - cgs units.  Wavelengths in micron.  Plain pointers and sizes only; no C++ types.
 *  - Every call returns mcrt_status (0 = ok, < 0 = error) and never aborts or throws.  The text of
 *    the last error of a context is available from mcrt_last_error().
 *  - The caller owns every pointer it passes.  The library copies during the call and never keeps
 *    a caller pointer.  Outputs are written into caller-allocated buffers.  A buffer tagged
 *    MCRT_DEVICE is device memory on the current CUDA device (e.g. torch.Tensor.data_ptr()).
 *  - The context owns the device memory it allocates; mcrt_destroy gives it back -- to a cache of
 *    the library (blocks of up to 256 MB, 1 GB in all, reused by the next context that asks for
 *    the same size, so that a second job of the same shape allocates nothing);
 *    mcrt_release_cached_memory() returns the cache to the driver.  A context may be destroyed
 *    with any device current.
 *  - Call order: mcrt_grid_create -> mcrt_set_opacity -> mcrt_set_source -> mcrt_run_batch (any
 *    number) -> getters.  A call out of order returns MCRT_ESTATE.
 *  - All arithmetic of the method runs in CUDA kernels on an sm_100a device.  There is no CPU
 *    fallback: without a usable device every call that needs one returns MCRT_ECUDA.
 *  - Determinism: results depend only on (grid, opacity, sources, seed, the sequence of
 *    (first_packet_id, n_packets) batches), never on thread scheduling: temperatures are frozen
 *    within a batch, every packet owns the Philox4x32-10 stream keyed by (seed, packet id), and
 *    all tallies are integers.
 */
#ifndef MCRT_H_
#define MCRT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mcrt_ctx mcrt_ctx; /* opaque */

typedef enum {
  MCRT_OK = 0,
  MCRT_EINVAL = -1, /* NULL pointer, bad size, source outside the grid, ... */
  MCRT_ESTATE = -2, /* call out of order */
  MCRT_ENOMEM = -3, /* host or device allocation failed */
  MCRT_ECUDA = -4   /* CUDA runtime error or no usable device; see mcrt_last_error */
} mcrt_status;

typedef enum { MCRT_HOST = 0, MCRT_DEVICE = 1 } mcrt_mem;

/* ---- grid ("cubes ... further divided into subcubes (cells)") ------------------
 * Root grid of n_root^3 cubes, x fastest.  A cube flagged in `refine` is divided into sub^3
 * subcubes.  Leaf slots (layout R22), used by every per-cell getter:
 *   slot = ix + n_root*(iy + n_root*iz)                      for an unrefined cube,
 *   slot = n_root^3 + sub^3*k + (sx + sub*(sy + sub*sz))     for a subcube of the k-th refined
 *                                                            cube (k counts flagged cubes in
 *                                                            x-fastest order);
 * the slot of a refined root cube itself is unused (density 0, tally 0, T = T_min).
 * Densities that are negative or NaN are taken as 0. */
typedef struct {
  int32_t n_root;        /* N >= 1; N^3 + n_ref*sub^3 must be < 2^31                          */
  int32_t sub;           /* S: 0 or 1 = no refinement, else 2..8 subcubes per edge            */
  double origin[3];      /* cm, low corner of the box                                         */
  double root_size;      /* cm, edge of a root cube, > 0                                      */
  const uint8_t* refine; /* [N^3] 1 = cube is subdivided; NULL = none                         */
  const float* rho_root; /* [N^3] g cm^-3 of dust; ignored where refine = 1                   */
  const float* rho_sub;  /* [n_ref*S^3]; NULL iff no cube is refined                          */
  mcrt_mem mem;          /* where refine / rho_root / rho_sub live                            */
  int32_t layout;        /* device storage order of the root grid (never visible in the getters,
                            which always use the slot order above): 0 = automatic, 1 =
                            x-fastest, 2 = 8^3 bricks in Morton order (automatic for a
                            single-level grid larger than the L2), 3 / 4 = macro cubes of 4^3 /
                            8^3 cells: a single-level grid run internally as a two-level one in
                            which a cube of cells that all hold the same density is crossed in
                            one step (on request only; n_root must be a multiple of 4 / 8: it
                            pays where flights cross many uniform cubes, e.g. an optically thin
                            sphere in vacuum -- DESIGN.md section 6).
                            Subcubes always follow the root grid as blocks of sub^3.           */
} mcrt_grid_desc;

/* Creates a context on the current CUDA device and uploads the grid. */
mcrt_status mcrt_grid_create(const mcrt_grid_desc* desc, mcrt_ctx** out);
mcrt_status mcrt_destroy(mcrt_ctx* ctx);
/* Number of leaf slots = length of every per-cell array.  < 0 on a NULL context. */
int64_t mcrt_leaf_slots(const mcrt_ctx* ctx);

/* ---- opacity (cross-sections per dust component and abundances) -------------
 * n_bins frequency bins given by n_bins+1 ascending wavelength edges (R4); bin centre = geometric
 * mean of its edges; a packet's frequency is a bin index.  The species are mixed by mass weight
 * into one grain with one temperature per cell (R13).  The library builds, in fp64 kernels and
 * stored as fp32: mixed kappa_ext, albedo, g; Q(T_k) = sum_j kappa_abs,j B_j(T_k) dnu_j on
 * T_k = T_min (T_max/T_min)^(k/(n_T-1)); and the emission inverse-CDF rows C_k[j] (midpoint rule,
 * R5; PAPER.md L27 Eqn 11.67).  All pointers are HOST pointers (the tables are small). */
typedef struct {
  int32_t n_bins;                /* 1..4096; 32*n_bins + 24*n_root bytes of shared memory per
                                    block must stay below 227 KB (else MCRT_EINVAL)            */
  const double* lambda_edges_um; /* [n_bins+1] ascending, > 0                                 */
  int32_t n_species;             /* >= 1                                                      */
  const double* weight;          /* [n_species] mass fractions                                */
  const float* kabs;             /* [n_species][n_bins] cm^2 g^-1                             */
  const float* ksca;             /* [n_species][n_bins] cm^2 g^-1                             */
  const float* g;                /* [n_species][n_bins] <cos theta> of Henyey-Greenstein      */
  double T_min, T_max;           /* K; temperature table range                                */
  int32_t n_T;                   /* rows; 0 = defaults T_min 1 K, T_max 1e4 K, n_T 801 (R11)  */
} mcrt_opacity_desc;
mcrt_status mcrt_set_opacity(mcrt_ctx* ctx, const mcrt_opacity_desc* desc);

/* ---- sources ("The star emits photon packages of constant energy") -------------
 * type 0: isotropic point source at pos (must lie inside the box, else MCRT_EINVAL);
 * type 1: external isotropic field entering through the six box faces (R25), pos ignored.
 * Each source radiates a blackbody spectrum of temperature T_bb truncated to the band (R6) with
 * in-band luminosity L.  A packet picks its source with probability L_s / sum L (R26).
 * Replaces all sources.  Host pointer. */
typedef struct {
  int32_t type;
  double pos[3]; /* cm */
  double L;      /* erg s^-1, > 0 */
  double T_bb;   /* K, > 0 */
} mcrt_source;
mcrt_status mcrt_set_source(mcrt_ctx* ctx, int32_t n_src, const mcrt_source* src);

/* ---- the hot path -----------------------------------------------------------
 * Transports packets first_packet_id .. first_packet_id + n_packets - 1 with the cell
 * temperatures frozen (emission, free-flight optical depth tau* = -ln xi, cell walk through
 * cubes/subcubes, scatter or absorb + re-emit at nu ~ kappa_nu B_nu(T_cell), escape into the SED),
 * then adds the batch to the cumulative tallies and updates every cell temperature from
 * radiative equilibrium: 4 pi rho_i V_i Q(T_i) = cum_i * L_tot / N_cum (R9).
 * Asynchronous on `cuda_stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream;
 * NULL = the legacy default stream); getters synchronise with it.  n_packets = 0 is allowed
 * (only the temperature update runs). */
mcrt_status mcrt_run_batch(mcrt_ctx* ctx, uint64_t seed, uint64_t first_packet_id,
                           uint64_t n_packets, void* cuda_stream);

/* ---- the same batch in two halves, for packet-sharded multi-GPU runs ("scales
 * almost linearly with the number of graphical processing units") -----------------------------
 * Within a batch packages are independent (frozen temperatures, per-packet Philox streams), so
 * rank r of G transports its own range of packet ids with mcrt_transport_batch (rows a1..a8: no
 * temperature update), the ranks sum their cumulative integer tallies (one all-reduce of
 * mcrt_get_cell_energy(MCRT_DEVICE) arrays, done by the caller, e.g. NCCL through
 * torch.distributed), and every rank calls mcrt_update_temperature with the summed tally
 * (DEVICE pointer, [leaf slots]) and the number of packages emitted so far by ALL ranks (row a9).
 * tally_sum = NULL uses the context's own tally and count, which makes
 * transport_batch + update_temperature(NULL) identical to mcrt_run_batch. */
mcrt_status mcrt_transport_batch(mcrt_ctx* ctx, uint64_t seed, uint64_t first_packet_id,
                                 uint64_t n_packets, void* cuda_stream);
mcrt_status mcrt_update_temperature(mcrt_ctx* ctx, const uint64_t* tally_sum, uint64_t n_cum,
                                    void* cuda_stream);

/* The same exchange with HALF the bytes and no layout conversion (what sharding.ShardedRunner uses):
 * mcrt_transport_batch_delta zeroes `delta_dev` (DEVICE, uint32[mcrt_delta_words], owned by the
 * caller, e.g. a torch int32 tensor: mcrt_store_slots words for the grains in equilibrium, followed --
 * once a PAH is declared (mcrt_set_pah) -- by mcrt_store_slots x n_bins words for the PAH's absorbed
 * spectrum of every leaf), then transports this rank's packets tallying the batch's
 * absorptions into it instead of into the cumulative tally; the ranks all-reduce (sum) their delta
 * arrays; mcrt_accumulate_update adds the summed delta to the context's cumulative tally and
 * updates the temperatures with n_cum = packages emitted so far by ALL ranks (one kernel).  The
 * array is in the library's internal STORAGE order (root grid possibly bricked and padded,
 * subcubes behind it): opaque to the caller, identical on every rank that created the same grid.
 * After the call every rank's mcrt_get_cell_energy returns the global cumulative counts. */
int64_t mcrt_store_slots(const mcrt_ctx* ctx);
int64_t mcrt_delta_words(const mcrt_ctx* ctx);
mcrt_status mcrt_transport_batch_delta(mcrt_ctx* ctx, uint64_t seed, uint64_t first_packet_id,
                                       uint64_t n_packets, uint32_t* delta_dev, void* cuda_stream);
mcrt_status mcrt_accumulate_update(mcrt_ctx* ctx, const uint32_t* delta_sum_dev, uint64_t n_cum,
                                   void* cuda_stream);

/* ---- results ("Each absorption event raises the energy of the cell by eps, and
 * accordingly its temperature"; L27, L31: the computed SED) ------------------------------------
 * n_abs_out[leaf slots]: cumulative number of packages absorbed per leaf (exact integers; "cell
 * energy" in units of eps, R23).  *eps_out (host pointer, may be NULL) = L_tot / N_cum in erg s^-1
 * per package, so that the absorbed power of a cell is n_abs * eps. */
mcrt_status mcrt_get_cell_energy(mcrt_ctx* ctx, uint64_t* n_abs_out, double* eps_out, mcrt_mem mem);
/* T_out[leaf slots] in K; T_min for cells that absorbed nothing or hold no dust. */
mcrt_status mcrt_get_cell_temperature(mcrt_ctx* ctx, float* T_out, mcrt_mem mem);
/* The temperatures of mcrt_get_cell_temperature(ctx, T_out, MCRT_HOST), read out WITHOUT allocating
 * device memory.  Who needs it: the ordinary getter converts the stored temperature rows to kelvin
 * in slot order (R22) with a kernel, and that kernel needs a device array to write to before the
 * copy to the host -- the getter cudaMallocs one (4..8 B x leaf slots) the first time it is used
 * on a context.  Some callers must not, or cannot, do that between batches: a process whose
 * device memory is already handed out in full to another allocator (a torch caching pool, a fixed
 * MPS / MIG memory quota) where a late cudaMalloc fails; a host thread that runs while another
 * thread of the process records a CUDA graph in global capture mode, where any cudaMalloc breaks
 * the recording; a latency-bound control loop that cannot afford the device-wide synchronisation
 * a cudaMalloc or cudaFree may imply.  For them the conversion kernel of this call writes into an
 * array that is part of the library image: MCRT_NOALLOC_MAX_SLOTS floats (4 MiB), which every GPU
 * that loads libmcrt.so holds from load until the process exits, used or not.
 *   T_out: HOST pointer, [leaf slots] floats, owned by the caller; K, same values bit for bit as
 *     the ordinary getter's.  The call returns after the copy to T_out has completed.
 *   Limit: mcrt_leaf_slots(ctx) <= MCRT_NOALLOC_MAX_SLOTS, else MCRT_EINVAL and a message naming
 *     both numbers (C0 and C1 fit; the disks and the 512^3 cube do not: use the ordinary getter).
 *   The context's device must be the current device (MCRT_ESTATE otherwise).
 *   The first call on a GPU asks the driver once where that GPU's copy of the array lives
 *     (cudaGetSymbolAddress); later calls reuse the answer.  Make that first call before any
 *     stream capture starts.
 *   The call makes no cudaMalloc, cudaFree or other allocating CUDA call, and nothing is freed.
 *   ONE array per GPU serves every context and every call, and it keeps whatever the previous call
 *     left in it.  Nothing has to be cleared: each of the [leaf slots] floats copied out is written
 *     by this call's kernels first, and no float beyond them is read.  Two such calls in flight on
 *     one GPU at the same time would overwrite each other's temperatures; the library therefore
 *     takes a process-wide lock for the whole call and does not return before its copy is done.
 *     Do not work around that (e.g. by copying the array yourself from another stream). */
#define MCRT_NOALLOC_MAX_SLOTS 1048576
mcrt_status mcrt_get_cell_temperature_noalloc(mcrt_ctx* ctx, float* T_out_host);
/* counts_out[3][n_bins]: escaped packages per bin; component 0 = direct (never interacted),
 * 1 = scattered only, 2 = thermal (re-emitted at least once) (R24). */
mcrt_status mcrt_get_sed(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem);

typedef struct {
  uint64_t emitted, escaped, lost, absorptions, scatterings, flights, crossings;
} mcrt_counters;

/* ---- all results of a batch in one call, optionally overlapped with the next batch -------------
 * The getters above synchronise once each.  mcrt_get_results reads any subset of the same arrays
 * (cell energies and temperatures; L27, L31: the SED) with ONE synchronisation;
 * mcrt_results_begin only queues the read-out and returns a ticket (0 or 1; two may be in flight):
 * on the stream of the last batch it snapshots what was asked for (slot order, R22) into buffers
 * the context owns, then copies the snapshot to the caller's buffers on a stream of its own, so a
 * mcrt_run_batch issued right after it overlaps the transfer; mcrt_results_wait(ticket) blocks
 * until that ticket's buffers are filled.  `mem` says where n_abs / T / sed / emitted_per_bin
 * live (MCRT_HOST buffers should be pinned for the copies to overlap); counters and eps are host
 * pointers always.  Any member may be NULL.  The buffers must stay valid until the wait. */
typedef struct {
  uint64_t* n_abs;           /* [leaf slots] cumulative absorbed packages per leaf             */
  float* T;                  /* [leaf slots] K                                                  */
  uint64_t* sed;             /* [3][n_bins]                                                     */
  uint64_t* emitted_per_bin; /* [n_bins]                                                        */
  mcrt_counters* counters;   /* host                                                            */
  double* eps;               /* host: L_tot / N_cum                                             */
} mcrt_results;
mcrt_status mcrt_get_results(mcrt_ctx* ctx, const mcrt_results* out, mcrt_mem mem);
mcrt_status mcrt_results_begin(mcrt_ctx* ctx, const mcrt_results* out, mcrt_mem mem, int32_t* ticket);
mcrt_status mcrt_results_wait(mcrt_ctx* ctx, int32_t ticket);
/* Cumulative event counters (host struct) and, if not NULL, emitted packages per bin
 * (host, [n_bins]).  `crossings` counts every exit of a packet from a leaf through a face,
 * including the final exit from the box (R27).  `lost` counts packets dropped at the flight cap
 * of 10^7 (R20) and must be 0. */
mcrt_status mcrt_get_counters(mcrt_ctx* ctx, mcrt_counters* out, uint64_t* emitted_per_bin);
/* what: bit 0 = SED + counters, bit 1 = cell energy + temperatures + N_cum. */
mcrt_status mcrt_reset_tallies(mcrt_ctx* ctx, int32_t what);

/* ---- direction-resolved output (the paper's product is an 11.3 um image and
 * flux profiles; reading R34) ---------------------------------
 * Escaping packages are additionally binned by their direction:
 *  - inclination: mu = d_z in n_mu bins uniform over [-1, 1]; counts [n_mu][3][n_bins] with
 *    the components of mcrt_get_sed; summing over mu gives mcrt_get_sed exactly.
 *  - image: packages of the bins bin_lo..bin_hi (bin_hi < 0 = last bin) that leave within
 *    half_angle_deg of the direction `dir` (pointing from the grid TOWARDS the observer) are
 *    binned by their impact vector b = r - (r.d) d (r = position relative to the box centre,
 *    d = direction of flight) on the orthonormal image axes e1 = z x dir normalised (within
 *    2.6 degrees of the z axis: the component of x normal to dir, normalised) and e2 = dir x e1: n_pix x n_pix pixels over [-half_width, half_width]^2 cm, row index along
 *    e2, column index along e1; counts [n_pix][n_pix].
 * n_mu = 0 / n_pix = 0 switch the respective tally off.  Needs the opacity (n_bins); calling
 * mcrt_set_opacity again switches the observer off.  Setting an observer zeroes its tallies;
 * mcrt_reset_tallies(bit 0) zeroes them too. */
typedef struct {
  int32_t n_mu;
  int32_t n_pix;
  double dir[3];
  double half_angle_deg;   /* (0, 180]                                                       */
  double half_width;       /* cm, > 0                                                        */
  int32_t bin_lo, bin_hi;
} mcrt_observer_desc;
mcrt_status mcrt_set_observer(mcrt_ctx* ctx, const mcrt_observer_desc* desc);
mcrt_status mcrt_get_sed_mu(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem);
mcrt_status mcrt_get_image(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem);

/* ---- transiently heated PAH (the method is "extended to the treatment of transiently
 * heated PAHs"; L45 Fig. 3: their temperature distribution P(T); L49: "P(T) depends strongly on the
 * hardness and spectral shape of the exciting radiation field"; DESIGN.md
 * readings R35..R40 -- the paper prints no formula, the cited book and the PAH data are not
 * available) ------------------------------------------------------------------------------------
 * One PAH kind per context, declared AFTER mcrt_set_opacity as a part of that dust mix:
 * kabs_pah[n_bins] = absorption of the PAH in cm^2 per gram of the MIX (clipped to the mix's
 * kappa_abs).  The grains in equilibrium keep the rest: Q(T) and the emission rows are rebuilt
 * from it.  From then on an absorbed package is taken by the PAH with probability kappa_PAH,j /
 * kappa_abs,j (R36); it is booked on the leaf's absorbed spectrum (per leaf and bin) and
 * re-emitted from the leaf's PAH emission spectrum.  After every batch each leaf's absorbed
 * spectrum gives the photon absorption rates of one molecule (R40: counts * L_tot / N_cum / h nu /
 * molecules in the leaf, a molecule = n_C carbon atoms, the PAH hold mass_fraction of the dust
 * mass), its stationary temperature distribution P(T_k) on n_Tp log-spaced temperatures (R38:
 * enthalpy U(T) = 3 n_C k theta (x - atan x), x = T/theta (R37); photon jumps shared linearly
 * between the two bracketing states; cooling to the next lower state at the rate
 * 4 pi sum_j C_j B_j(T) dnu_j / (U_k - U_k-1)), and the emission CDF sum_k P_k C_j B_j(T_k) dnu_j
 * (R39).  n_Tp = 0 takes the defaults 128 states, 5 K .. 1e4 K; theta_K <= 0 takes 500 K.
 * Calling mcrt_set_opacity again drops the PAH; mcrt_reset_tallies(bit 1) zeroes its tallies.
 * Host pointers.  Packet-sharded batches carry the PAH's tallies in the same delta array (mcrt_delta_words). */
typedef struct {
  int32_t n_C;            /* carbon atoms per molecule, >= 1                                    */
  double mass_fraction;   /* of the dust mass, (0, 1]                                           */
  const float* kabs_pah;  /* [n_bins] cm^2 per gram of the dust mix                             */
  double theta_K;         /* temperature scale of the enthalpy law                              */
  double T_lo, T_hi;      /* K: range of the states                                             */
  int32_t n_Tp;           /* number of states, 4..1024 (0 = defaults)                           */
} mcrt_pah_desc;
mcrt_status mcrt_set_pah(mcrt_ctx* ctx, const mcrt_pah_desc* desc);
/* counts_out[leaf slots][n_bins]: packages absorbed by the PAH per leaf and bin, cumulative (they
 * are NOT in mcrt_get_cell_energy, which counts the grains in equilibrium; the counter
 * `absorptions` counts both). */
mcrt_status mcrt_get_pah_absorbed(mcrt_ctx* ctx, uint32_t* counts_out, mcrt_mem mem);
/* cdf_out[leaf slots][n_bins]: the emission CDF the PAH of each leaf re-emits from in the next batch. */
mcrt_status mcrt_get_pah_emission_cdf(mcrt_ctx* ctx, float* cdf_out, mcrt_mem mem);
/* P(T) of the PAH of one leaf from its tallies so far: P_out[n_Tp] on the temperatures T_out[n_Tp]
 * (host pointers; T_out may be NULL). */
mcrt_status mcrt_get_pah_temperature_distribution(mcrt_ctx* ctx, int64_t leaf_slot, double* T_out, double* P_out);

/* Frees the device blocks the library keeps cached after contexts were destroyed (all devices);
 * returns the number of bytes given back to the driver.  Live contexts are not touched.  Call it
 * when another allocator of the process (torch, NCCL, your own cudaMalloc) needs the memory. */
int64_t mcrt_release_cached_memory(void);
/* Text of the last error: of the context, or -- with NULL -- of the last call of the calling
 * thread that failed without a context (mcrt_grid_create, the context-free calls of mcrt_dev.h). */
const char* mcrt_last_error(const mcrt_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MCRT_H_ */
