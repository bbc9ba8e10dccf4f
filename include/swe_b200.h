/* swe_b200.h -- C ABI of the B200-native shallow-water time-step library.
 *
 * What it computes: the explicit finite-volume time step of Delmas & Soulaimani,
 * "Parallel high-order resolution of the Shallow-water equations on real large-scale meshes with
 * complex bathymetries" (arxiv 2307.16758; citations below are PAPER.md:<line>), section 6.1-6.2,
 * on an unstructured triangle mesh, in fp64, on ONE NVIDIA B200 (sm_100a):
 *   eq. 1   state U=(h, hu, hv)
 *   eq. 2   rotational invariance F.n = T^-1 G(T U)
 *   eq. 3   finite-volume update over the three sides of a triangle
 *   BCs     transmissive / imposed inflow Q / wall (Q=0)
 *   eq. 5   CFL time step, d = radius of the inscribed circle
 *   eq. 6-14  HLL / HLLC flux and wave-speed estimates
 *   eq. 15-21 WAF flux, TVD weights, SUPERBEE A(r,c)
 *   eq. 24-25 limiter semantics (beta=1 MINBEE) of the MUSCL slopes
 *   hydrostatic reconstruction, bed-slope S_O and friction S_f sources (named at PAPER.md:281,
 *   295, 422; formulas = DESIGN.md readings R12, R15); least-squares gradients and Heun RK2 for
 *   MUSCL (BASELINE.json north_star); ghost layers, send list + contiguous receive range per
 *   neighbour, send buffer refreshed on the GPU every step          PAPER.md:121-127, 141, 460.
 *
 * Conventions (every entry point):
 *   - returns SWE_OK (0) or a negative SWE_ERR_* code; never throws across the ABI; the message of
 *     the last failure on the calling thread is returned by swe_last_error();
 *   - array arguments are caller-owned and only read (inputs) or written (outputs) during the
 *     call; every array pointer may be a HOST pointer or a DEVICE pointer of the current CUDA
 *     device (classified with cudaPointerGetAttributes), so a torch tensor's data_ptr() can be
 *     passed straight through; outputs are caller-allocated with the stated length;
 *   - the user's cell numbering (the order of `tri`) is preserved at the boundary: the internal
 *     renumbering (space-filling curve) is invisible;
 *   - all real data are IEEE double, all indices int32 (counts int64);
 *   - there is no CPU fallback: without a CUDA device swe_mesh_create fails with SWE_ERR_CUDA.
 */
#ifndef SWE_B200_H
#define SWE_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swe_ctx swe_ctx; /* opaque; owns every host and device allocation it makes */

enum { SWE_OK = 0, SWE_ERR_ARG = -1, SWE_ERR_MESH = -2, SWE_ERR_CUDA = -3, SWE_ERR_STATE = -4,
       SWE_ERR_NOMEM = -5 };
/* scheme: first-order HLLC + Euler (eq. 6-14); MUSCL = least-squares gradients +
 * cell limiter + HLLC + Heun RK2 (north_star); WAF + Euler (eq. 15-21); MUSCL_MS = the paper's own
 * multislope MUSCL, eq. 22-25 PAPER.md:396-420 (upwind-average slopes, beta limiter: beta = 1
 * MINBEE, 2 SUPERBEE) + HLLC + Heun RK2 (reading R17). */
enum { SWE_HLLC = 0, SWE_MUSCL = 1, SWE_WAF = 2, SWE_MUSCL_MS = 3 };
/* boundary kinds (fixed level: PAPER.md:518, 548, reading R11) */
enum { SWE_BC_WALL = 0, SWE_BC_INFLOW_Q = 1, SWE_BC_LEVEL = 2, SWE_BC_TRANSMISSIVE = 3 };
/* cell renumbering for gather locality (north_star): Hilbert curve through the centroids, or reverse
 * Cuthill-McKee over the edge adjacency.  Results do not depend on it (orientation by user id). */
enum { SWE_RENUM_NONE = 0, SWE_RENUM_HILBERT = 1, SWE_RENUM_RCM = 2 };

/* Build the mesh (host: topology + geometry of SURVEY.md Appendix A.1, renumbering; then upload).
 *   nv, x, y, zb : vertices, coordinates [m] and bed elevation [m] per vertex
 *   nt, tri      : 3*nt vertex ids, any winding (re-oriented counter-clockwise internally)
 *   nb, bedge, btag : nb tagged boundary edges as 2*nb vertex ids + nb tag ids (>=0); boundary edges
 *                  not listed are walls.  Pointers may be NULL when nb == 0.
 *   renumber     : SWE_RENUM_*
 *   cuda_stream  : cudaStream_t the context will launch on (NULL = the legacy default stream)
 * Errors: SWE_ERR_ARG (NULL / negative sizes), SWE_ERR_MESH (vertex id out of range, zero-area
 * triangle, edge shared by more than two triangles, tagged edge that is not a boundary edge),
 * SWE_ERR_CUDA (no device / allocation or copy failure).  Initial state: h = hu = hv = 0, t = 0.
 * Defaults: g = 9.81, h_dry = 1e-6, h_thin = 1e-3, beta = 1, Manning n = 0, every tag = wall. */
int swe_mesh_create(swe_ctx** out, int64_t nv, const double* x, const double* y, const double* zb,
                    int64_t nt, const int32_t* tri, int64_t nb, const int32_t* bedge,
                    const int32_t* btag, int renumber, void* cuda_stream);
int swe_mesh_destroy(swe_ctx* ctx);
/* any output pointer may be NULL.  min_inradius: eq. 5's d. */
int swe_mesh_info(const swe_ctx* ctx, int64_t* ncell, int64_t* nedge, int64_t* nbedge,
                  double* min_inradius);
/* g [m/s2]; h_dry: wet threshold (wet <=> h > h_dry); h_thin: WAF falls back to HLLC within one
 * cell of depth <= h_thin (reading R14); beta: limiter parameter, kappa = beta/2 (1 = minmod /
 * MINBEE eq. 24, 2 = Barth-Jespersen, <= 0 = unlimited).  h_dry must be >= 1e-290: the kernels'
 * reciprocal / square-root sequences need every wet depth to be a normal fp64 number.
 * Errors: SWE_ERR_ARG (g <= 0, negative or NaN thresholds, h_dry < 1e-290). */
int swe_set_params(swe_ctx* ctx, double g, double h_dry, double h_thin, double beta);
/* Manning n per cell, length nt, user order; NULL = 0 everywhere (no friction). */
int swe_set_manning(swe_ctx* ctx, const double* n_cell);
/* kind of the boundary edges carrying `tag` and its value: discharge Q [m3/s, into the domain,
 * spread uniformly over the tag's total width] for SWE_BC_INFLOW_Q, free-surface level [m] for
 * SWE_BC_LEVEL; ignored otherwise. */
int swe_set_bc(swe_ctx* ctx, int tag, int kind, double value);
/* state, nt values each, user order.  SWE_ERR_STATE if any h is NaN or negative (the state is then
 * left as it was).  The simulated time t is not touched; use swe_set_time. */
int swe_set_state(swe_ctx* ctx, const double* h, const double* hu, const double* hv);
int swe_get_state(const swe_ctx* ctx, double* h, double* hu, double* hv);
/* swe_get_state for callers that must not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same result -- h, hu, hv of every cell, user order,
 * host or device pointers -- but host arrays are staged through a file-scope static device array
 * of 3 x SWE_STATIC_MAX_CELLS doubles (6 MiB, held by every GPU that loads the library until the
 * process exits) instead of a buffer that swe_get_state cudaMallocs on first use.  The call makes
 * no cudaMalloc / cudaFree and calls no allocating library routine; it launches the same kernel
 * on the context's stream and synchronises that stream before returning.  The device address of the
 * array is looked up once per device in swe_mesh_create (cudaGetSymbolAddress, with that device
 * current); the context's device must be current here too.
 * Limits: meshes of more than SWE_STATIC_MAX_CELLS cells are refused (SWE_ERR_ARG, message names
 * both numbers).  EVERY context on a device shares the one array and it keeps the last call's
 * contents: every slot a call copies out it has written first, so nothing needs clearing, but two
 * calls that overlap on the GPU (two contexts on different streams, two host threads) race on it --
 * serialise them.  Errors: SWE_ERR_ARG (NULL array, mesh too large), SWE_ERR_STATE (another device
 * is current), SWE_ERR_CUDA (no device address for the array; a CUDA failure). */
#define SWE_STATIC_MAX_CELLS 262144
int swe_get_state_static(const swe_ctx* ctx, double* h, double* hu, double* hv);
int swe_set_time(swe_ctx* ctx, double t);
/* Advance nsteps time steps: per step dt = cfl * min_i R_i/lambda_i (eq. 5) by a device
 * min-reduction, then the scheme's stage(s).  Asynchronous on the context's stream (dt never
 * visits the host) unless t_out or last_dt_out is non-NULL (host pointers), in which case the
 * call synchronises the stream and returns the simulated time and the last dt.  With zones built
 * (swe_zones_create) the step runs zone-wise with pack/unpack of the ghost cells every stage.
 * Errors: SWE_ERR_ARG (nsteps < 0, cfl <= 0, unknown scheme), SWE_ERR_STATE (zones built with too
 * few ghost layers for the scheme: WAF and MUSCL_MS need 2), SWE_ERR_CUDA. */
int swe_step(swe_ctx* ctx, int nsteps, double cfl, int scheme, double* t_out, double* last_dt_out);

/* swe_step replays one captured CUDA graph per time step when nsteps >= 2 (the step is a fixed
 * sequence of 3-11 kernels whose only varying input, dt, lives in device memory; on meshes below
 * ~1 M cells the step is launch-bound).  on = 0 launches the kernels one by one (default: on).  The
 * results are identical either way. */
int swe_set_graphs(swe_ctx* ctx, int on);

/* Cells without water are not worked on (wet/dry treatment of SURVEY.md section 8(c), A.3.5 /
 * A.6: a cell whose record is (0, 0, 0, z) has zero gradients, and an interior edge between two
 * such cells a zero flux record).  On the un-zoned mesh swe_step keeps one bit per cell / edge for
 * "this record holds nothing" (state buffers, gradient buffer, flux buffer; 0.5 bytes per cell in
 * all) and neither rewrites nor rereads such records from one stage to the next; a cell that is
 * (0, 0, 0, z) with three zero flux records is left as it is.  The results are bit-identical to the
 * step that works on every cell (on = 0, the default).  The bits are rebuilt by the first step
 * after any other call that may touch the buffers.  Opt-in because it pays only on meshes with
 * large dry areas, and less than the bytes it saves: on configs[3] the step
 * moves 22 % fewer bytes and takes 5 % less time; with every cell wet it costs 4-5 %. */
int swe_set_dry_masks(swe_ctx* ctx, int on);

/* Zone decomposition resident on this GPU.
 *   nzones : number of zones; zone_of_cell (nt, user order, values in [0,nzones)) or NULL =
 *            recursive coordinate bisection (nzones must then be a power of two)
 *   nlayers: ghost layers per zone, 1..3 (edge adjacency)
 * Each zone gets its own copy of its owned + ghost cells; per (zone, source zone) one send list
 * (indices into the source zone) and one contiguous receive range.  nzones == 0 removes zones.
 * The ghost layers and their numbering (sections 3.2-3.3)
 * are generated on the device: the layers of all zones grow together as bit masks over the edge
 * adjacency, one launch per layer, and a radix sort of (zone, source zone, layer, cell) keys gives
 * the contiguous receive ranges (csrc/swe_zone_kernels.cuh); the zones' own copies of connectivity
 * and geometry in that numbering are then gathered on the device as well
 * (csrc/swe_zone_assembly.cuh): the concatenated zoned mesh never exists on the host. */
int swe_zones_create(swe_ctx* ctx, int nzones, int nlayers, const int32_t* zone_of_cell);
/* wall-clock milliseconds of the last swe_zones_create / swe_zones_create_dist (host pointers,
 * any may be NULL): the device ghost-layer generation alone; the call up to and including the
 * host's link / exchange lists; the whole call.  SWE_ERR_STATE without zones. */
int swe_zone_setup_ms(const swe_ctx* ctx, double* ghost_layers_ms, double* build_ms, double* total_ms);
/* The same call broken down (host pointer, 5 doubles, milliseconds): [0] the zone of every cell
 * (recursive coordinate bisection, or mapping the caller's array), [1] the ghost layers of all
 * zones (device), [2] owned-cell positions (device) + links, send lists and per-rank exchange lists
 * (host, O(ghost cells)), [3] the zones' copies of connectivity and geometry assembled on the device
 * (swe_zone_assembly.cuh; section 3.3), [4] the whole call. */
int swe_zone_setup_detail(const swe_ctx* ctx, double* ms);
/* pack: send buffer[k] = U[send_idx[k]] for every link whose SOURCE is `zone` (-1 = all zones);
 * unpack: copy the buffers into the contiguous ghost ranges of `zone` (-1 = all). */
int swe_pack_ghosts(swe_ctx* ctx, int zone);
int swe_unpack_ghosts(swe_ctx* ctx, int zone);
int swe_zone_stats(const swe_ctx* ctx, int64_t* send_cells_total, int64_t* bytes_per_exchange,
                   int64_t* ghost_cells_total);
/* description of one zone for tests and for a multi-GPU driver: counts, then the arrays.
 * cells: user ids of owned cells then ghost blocks (nowned+nghost); layer: 0 owned, l = ghost
 * layer; links (one per source zone, ascending): src zone, receive start, count; send list of a
 * link = source-zone-local indices.  swe_zone_cells serves the zones resident on this rank (the
 * lists live on the device and are fetched the first time it is called); counts and links are
 * known for every zone.  Errors: SWE_ERR_ARG (no zones, no such zone, zone on another rank). */
int swe_zone_describe(const swe_ctx* ctx, int zone, int64_t* nowned, int64_t* nghost, int64_t* nlinks);
int swe_zone_cells(const swe_ctx* ctx, int zone, int32_t* cells, int32_t* layer);
int swe_zone_links(const swe_ctx* ctx, int zone, int32_t* src, int32_t* start, int32_t* count);
int swe_zone_sendlist(const swe_ctx* ctx, int zone, int link, int32_t* send_idx);

/* ---- zones distributed over ranks: one process per GPU (scope row f3) -------
 * The paper runs one MPI rank + one GPU per sub-domain and exchanges the ghost cells of U every
 * step.  Here rank r of nranks holds the zones [zone_begin[r], zone_begin[r+1])
 * of the SAME decomposition every rank builds from the same mesh (so no set-up message is needed:
 * each rank derives its own lists and its peers' independently, in the same order).  The library
 * never calls a communication library: the caller (paper_2307_16758_b200/dist.py, over
 * torch.distributed) moves or synchronises, the library packs, pushes and unpacks.  Per step:
 *     exchange(buffer 0); swe_dist_local_min -> all-reduce(min) -> swe_dist_begin_step;
 *     swe_dist_stage(scheme, 0); [Heun schemes: exchange(buffer 1); barrier; swe_dist_stage(scheme, 1)]
 * with exchange = swe_halo_push (peer memory, one kernel) or swe_halo_pack -> transfer ->
 * swe_halo_unpack.  swe_step refuses (SWE_ERR_STATE) while the zones are distributed.
 * swe_set_state / swe_set_manning / swe_set_bc are called on every rank with the same full-mesh
 * arguments; swe_get_state writes only the cells owned by this rank's zones and leaves the other
 * entries of the output arrays untouched.  nlayers >= 2 is required for MUSCL, WAF and MUSCL_MS
 * (no gradient exchange between ranks); nlayers = 1 serves HLLC.  Removing the zones again
 * (swe_zones_create(ctx, 0, ..)) brings back only the cells this rank owned: call swe_set_state with
 * the gathered full state before stepping un-zoned.
 *   zone_begin : nranks+1 non-decreasing zone ids from 0 to nzones (host pointer); may be NULL when
 *                nranks == 1.  Errors: SWE_ERR_ARG. */
int swe_zones_create_dist(swe_ctx* ctx, int nzones, int nlayers, const int32_t* zone_of_cell,
                          int nranks, int rank, const int32_t* zone_begin);
/* cells this rank sends to / receives from each peer per exchange (nranks entries each, host
 * pointers, either may be NULL); the halo buffers below hold 3 doubles (h, hu, hv) per cell, the
 * block of peer p starting at 3 * (sum of the counts of the peers before it). */
int swe_halo_counts(const swe_ctx* ctx, int64_t* send_cells, int64_t* recv_cells);
/* a10 across ranks: gather the send cells of state buffer `buffer` (0 = U / stage-1 input,
 * 1 = the Heun stage buffer U') into sendbuf (device pointer, 3 * total send cells doubles),
 * ordered by peer, then by (destination zone, source zone), then by position in the link. */
int swe_halo_pack(swe_ctx* ctx, int buffer, double* sendbuf);
/* copy recvbuf (device pointer, same ordering seen from the receiving side) into the contiguous
 * ghost ranges of `buffer`, then refresh the ghosts fed by zones resident on this rank. */
int swe_halo_unpack(swe_ctx* ctx, int buffer, const double* recvbuf);
/* Exchange over peer memory (NVLink / NVSwitch peer stores; PAPER.md:460's send buffer + in-place
 * receive fused into ONE kernel): swe_peer_export returns the CUDA IPC handles of this rank's two
 * state buffers (128 bytes: buffer 0 then buffer 1); the caller all-gathers them and calls
 * swe_peer_import(peer, handles of that peer) on every rank for every other rank.  Peers that live
 * in the same process (tests) are connected with swe_peer_raw / swe_peer_set_raw instead.
 * swe_halo_push(buffer) then stores every send cell's record straight into the ghost range of the
 * rank that needs it and refreshes the ghosts fed by resident zones.  It is asynchronous on the
 * context's stream and does NOT synchronise the ranks: before a rank reads its ghosts, every peer's
 * push must have completed, and before a push, the target must have finished reading the ghosts of
 * that buffer -- the caller orders this with a stream-ordered collective (the all-reduce of dt after
 * the push of buffer 0, a barrier after the push of buffer 1; dist.py).  Errors: SWE_ERR_STATE (no
 * zones / a peer with a non-empty send list not imported), SWE_ERR_CUDA (IPC failure). */
int swe_peer_export(swe_ctx* ctx, unsigned char* handles /* 128 bytes, host */);
int swe_peer_import(swe_ctx* ctx, int peer, const unsigned char* handles /* 128 bytes, host */);
int swe_peer_raw(swe_ctx* ctx, void** buf0, void** buf1);
int swe_peer_set_raw(swe_ctx* ctx, int peer, void* buf0, void* buf1);
int swe_halo_push(swe_ctx* ctx, int buffer);
/* a9 across ranks: min over this rank's owned wet cells of R_i / lambda_i (eq. 5), +inf if none,
 * written to min_out (DEVICE pointer, 1 double; no host synchronisation).  After the last stage of
 * a step the value is already there (folded into the update). */
int swe_dist_local_min(swe_ctx* ctx, double* min_out);
/* dt = cfl * (*min_in) (DEVICE pointer: the all-reduced minimum; +inf -> dt = 0, the step is a
 * no-op), t += dt. */
int swe_dist_begin_step(swe_ctx* ctx, const double* min_in, double cfl);
/* one stage of the scheme on this rank's zones: stage 0 reads buffer 0 (Heun: writes buffer 1;
 * Euler schemes: updates buffer 0 in place and end the step); stage 1 (Heun only) reads buffer 1
 * and writes U^{n+1} = (U^n + E(U'))/2 to buffer 0.  The ghosts of the buffer read must be current. */
int swe_dist_stage(swe_ctx* ctx, int scheme, int stage);
/* The two halves of swe_dist_stage, for the overlap schedule (scope row f2; "high
 * overlap": the cells of the send lists are updated first, the exchange runs while the rest of the
 * domain is updated).  swe_dist_flux: gradient + limiter (MUSCL) and edge fluxes of the stage's
 * input buffer.  swe_dist_update: the cell update of the stage for part 0 = every owned cell,
 * 1 = only the cells on a send list (remote or resident), 2 = every owned cell but those.  A stage
 * is flux, then part 0, or flux, part 1, part 2 (in that order: part 2 or 0 of the last stage ends
 * the step).  The results are bit-identical to swe_dist_stage. */
int swe_dist_flux(swe_ctx* ctx, int scheme, int stage);
int swe_dist_update(swe_ctx* ctx, int scheme, int stage, int part);
/* simulated time and last dt (host pointers; synchronises the stream). */
int swe_get_time(swe_ctx* ctx, double* t_out, double* last_dt_out);

/* ---- single passes of the hot path, exposed for parity tests and kernel timing -------------
 * (SURVEY.md section 8(a) rows a2, a3-a7, a8, a9).  They act on the current state, un-zoned. */
/* a9: dt = cfl * min over wet cells of R_i / (sqrt(g h) + |u|) (eq. 5); 0 if no wet cell. */
int swe_compute_dt(swe_ctx* ctx, double cfl, double* dt_out /* host */);
/* a2: limited least-squares gradients, out[8*nt], user order, per cell
 * (eta_x, eta_y, h_x, h_y, u_x, u_y, v_x, v_y). */
int swe_gradients(swe_ctx* ctx, double* out);
/* a3-a7: fluxes of the current state with time step dt (dt only matters for WAF): per cell and
 * local side k=0..2, sigma * Phi (3 components) as the cell sees it, out[9*nt], user order,
 * out[9*i + 3*k + c]; local side k joins vertices k -> k+1 of the counter-clockwise triangle. */
int swe_side_fluxes(swe_ctx* ctx, double dt, int scheme, double* out);
/* a8 (+a2..a7): one Euler stage with a given dt from the current state, result to caller arrays
 * (nt each, user order); the context's state is not changed. */
int swe_euler_stage(swe_ctx* ctx, double dt, int scheme, double* h1, double* hu1, double* hv1);
/* counters: steps taken, kernels launched by this context so far, bytes moved by pack+unpack. */
int swe_get_stats(const swe_ctx* ctx, int64_t* steps, int64_t* kernel_launches, int64_t* halo_bytes);
/* For a caller that captures a sequence of this context's calls into a CUDA graph of its own and
 * replays it (paper_2307_16758_b200/dist.py does so for the distributed step, collectives included):
 * adds the steps, kernel launches and halo bytes of the replays to the counters of swe_get_stats
 * (the library only sees the calls made during the capture).  Arguments may be negative (to take
 * the recorded-but-not-run capture pass out again).  Errors: SWE_ERR_ARG. */
int swe_account_replays(swe_ctx* ctx, int64_t steps, int64_t kernel_launches, int64_t halo_bytes);
/* time the hot path with CUDA events on the context's stream: runs swe_step(nsteps,...) between
 * two events and returns the elapsed milliseconds (synchronises). */
int swe_step_timed(swe_ctx* ctx, int nsteps, double cfl, int scheme, float* ms_out);
/* fp64 FMA throughput of the device in TFLOP/s (2 flops per FMA; eight independent chains per
 * thread, 8 blocks of 256 threads per SM, best of 3 timed launches): the ALU-side roofline the
 * bandwidth-bound claim is checked against.  Synchronises. */
int swe_fp64_peak(swe_ctx* ctx, double* tflops_out);

/* How much of the CURRENT state the dry-cell / dry-edge skips of the gradient and flux kernels
 * ("cells without water are not worked on") leave alone; bench.py prints the
 * fractions beside its roofline figures.  counts (host pointer, 5 entries): [0] owned cells that
 * are not wet (h <= h_dry), [1] owned cells with h == 0, [2] interior edges between two cells with
 * h == 0, [3] cells of the mesh, [4] interior edges of the un-zoned mesh.  With zones the edge count
 * [2] runs over the zoned copy (edges between ghost cells included).  Synchronises.
 * Errors: SWE_ERR_ARG, SWE_ERR_CUDA. */
int swe_dry_counts(const swe_ctx* ctx, int64_t* counts);

/* Test interface: the kernels' own division and square-root sequences (MUFU seed + one Newton step +
 * residual correction, swe_kernels.cuh) against the IEEE-rounded a[i] / x[i] and sqrt(x[i]) on n
 * caller-supplied samples (host or device pointers; x > 0, everything in the normal range).
 * ndiff[0], ndiff[1]: how many quotients / roots differ from the IEEE result; maxrel[0], maxrel[1]:
 * the largest relative difference of each.  Errors: SWE_ERR_ARG, SWE_ERR_CUDA. */
int swe_fastmath_check(swe_ctx* ctx, int64_t n, const double* a, const double* x, int64_t* ndiff, double* maxrel);
/* per-kernel timing: runs `reps` launches of one kernel of the hot path on the current state
 * between two events; which: 0 dt_reduce, 1 grad_limit (scheme SWE_MUSCL_MS: the multislope side
 * records, k_ms_slopes), 2 edge_flux(scheme), 3 cell_update (Euler
 * stage), 4 cell_update (Heun combine), 5 pack, 6 unpack.  The state is left unchanged (updates
 * write to the stage buffer). */
int swe_kernel_timed(swe_ctx* ctx, int which, int scheme, int reps, float* ms_out);

/* per-kernel timing inside swe_step: with profiling on, every kernel launch of swe_step is
 * bracketed by two CUDA events on the context's stream; swe_get_profile synchronises and returns
 * accumulated milliseconds and launch counts per kind (7 each):
 * 0 dt_reduce, 1 grad_limit (or the multislope side records), 2 edge_flux, 3 cell_update (both the
 * full and the send-list launches), 4 pack (and the peer-memory push), 5 unpack, 6 dt_finalize. */
int swe_set_profile(swe_ctx* ctx, int on);
int swe_get_profile(swe_ctx* ctx, double* ms, int64_t* count);

const char* swe_last_error(void); /* thread-local, static storage */

/* ---- host-only inspection of the set-up (no GPU needed; used by the CPU test-suite) ----------
 * swe_host_mesh_build runs the same host set-up as swe_mesh_create (topology, geometry of
 * SURVEY.md A.1, renumbering) and swe_host_zones_build the zone builder of A.12, without touching
 * a device.  swe_host_get copies a named array out (see csrc/host_inspect.cpp for the names) and
 * returns its element count (-1 capacity too small, -2 unknown name). */
int swe_host_mesh_build(void** out, int64_t nv, const double* x, const double* y, const double* zb,
                        int64_t nt, const int32_t* tri, int64_t nb, const int32_t* bedge,
                        const int32_t* btag, int renumber);
int swe_host_zones_build(void* handle, int nzones, int nlayers, const int32_t* zone_of_cell);
/* the distributed variant (swe_zones_create_dist's host half): adds the names "zone_rank",
 * "rsend_idx", "rsend_dst", "rsend_peer", "rrecv_idx", "rsend_off", "rrecv_off", "send_cells" to
 * swe_host_get. */
int swe_host_zones_build_dist(void* handle, int nzones, int nlayers, const int32_t* zone_of_cell,
                              int nranks, int rank, const int32_t* zone_begin);
void swe_host_mesh_free(void* handle);
int64_t swe_host_get(void* handle, const char* name, void* out, int64_t capacity_bytes);
const char* swe_host_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SWE_B200_H */
