/* mm.h - C ABI of the B200-native micromagnetic hot path (libmm_b200.so).
 *
 * What it computes (citations: Lnnn = line of PAPER.md, arXiv 1406.7635, "The design and
 * verification of MuMax3"; readings of silent/garbled passages are listed in DESIGN.md):
 *   B_eff = B_ext + B_demag + B_exch + B_anis                         (L108-L113)
 *   B_demag,i = K_ij * (mu0 Msat m_j), FFT-accelerated convolution     (Eq. 3)
 *   B_exch: 6-neighbour stencil with region look-up tables             (Eq. 6, Eq. 9)
 *   B_anis: uniaxial (Eq. 18) and cubic (Eq. 21)
 *   torque = -gamma/(1+alpha^2) [m x B + alpha m x (m x B)]            (Eq. 2)
 *   time stepping: Dormand-Prince RK45, FSAL, error eps = dt max|tau_hi - tau_lo|, adaptive dt
 *   with MaxErr and headroom 0.8                                       (L365, L372-L374)
 * All field arithmetic is fp32 on the GPU (L19, L143: "single precision"); the demag kernel is
 * built in fp64 and truncated to fp32 (L143); time and dt are fp64.
 *
 * Conventions
 *   - SI units: metres, A/m, J/m, J/m^3, tesla, seconds (as in the paper's scripts, L60-L66).
 *   - Arrays are structure-of-arrays [component][z][y][x], x fastest; N = Nx*Ny*Nz cells, so a
 *     vector field is 3N floats and the region map N bytes.
 *   - Every array argument may be a HOST pointer or a DEVICE pointer (told apart with
 *     cudaPointerGetAttributes). The caller owns every buffer it passes; the library copies
 *     during the call (the handle's stream is synchronised before an input call returns, for host
 *     and device sources alike) and keeps no reference. The handle owns its device memory.
 *   - All work is enqueued on the handle's CUDA stream: the one passed to mm_create_ex, or, if none
 *     was passed, a stream the handle creates for itself (a blocking stream: it stays ordered with
 *     work on the legacy default stream; mm_get_stream returns it). Calls that return data to the
 *     caller (mm_get_*, mm_b_eff, mm_step_rk45 with info != NULL, mm_run) synchronise that stream.
 *   - Every call returns MM_OK (0) or a negative error code; nothing throws or aborts across the
 *     ABI. mm_last_error() gives a text for the last failure on a handle.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - There is no CPU fallback: without a CUDA device mm_create fails with MM_ECUDA.
 */
#ifndef MM_B200_H
#define MM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mm_sim mm_sim; /* opaque handle */

enum { MM_OK = 0, MM_EINVAL = -1, MM_ENOMEM = -2, MM_ECUDA = -3, MM_ESTATE = -4, MM_ENAN = -5, MM_EDT = -6 };

/* terms of B_eff (L108-L113); a mask replaces the paper's EnableDemag switch (L611) */
enum { MM_DEMAG = 1, MM_EXCH = 2, MM_ANIS = 4, MM_ZEEMAN = 8, MM_ALL = 15 };

#define MM_MAX_REGIONS 256 /* "region index between 0 and 256", L43 */

/* Per-region material look-up tables (L43, Fig. 1) and the uniform applied field.
 * All doubles, SI; the library converts to fp32 tables on the device. Host memory only. */
typedef struct {
  int nregions;                     /* 1..256; region ids >= nregions in the map -> MM_EINVAL */
  double Msat[MM_MAX_REGIONS];      /* A/m, >= 0 (0 = vacuum: no torque, no exchange) */
  double Aex[MM_MAX_REGIONS];       /* J/m, >= 0 */
  double alpha[MM_MAX_REGIONS];     /* damping */
  double Ku1[MM_MAX_REGIONS];       /* J/m^3, Eq. 18 */
  double Ku2[MM_MAX_REGIONS];
  double anisU[MM_MAX_REGIONS][3];  /* uniaxial axis; normalised by the library */
  double Kc1[MM_MAX_REGIONS];       /* J/m^3, Eq. 21 */
  double Kc2[MM_MAX_REGIONS];
  double Kc3[MM_MAX_REGIONS];
  double anisC1[MM_MAX_REGIONS][3]; /* cubic axes c1, c2 (normalised); c3 = c1 x c2 (L286) */
  double anisC2[MM_MAX_REGIONS][3];
  double B_ext[3];                  /* uniform applied field, tesla */
  const double* exch_scale;         /* NULL => S = 1; else lower-triangular S[i(i+1)/2 + j], i >= j,
                                       nregions(nregions+1)/2 entries (Eq. 9) */
  double gamma_LL;                  /* rad/(T s); 0 => 1.7595e11 (L859) */
} mm_params;

typedef struct {
  double t;        /* simulation time after the attempt, s */
  double dt_taken; /* step size that was attempted */
  double dt_next;  /* controller's suggestion for the next attempt */
  double err;      /* eps = dt * max_cells || sum_j e_j tau_j ||_2   (L372) */
  int accepted;    /* 1 if the step was taken (always 1 with a fixed step) */
  long n_eval;     /* torque evaluations so far (the paper's Neval counter, L1071) */
} mm_step_info;

/* Create a simulation box (the paper's setgridsize / setcellsize / SetPBC, L60-L61, L175).
 * Nx,Ny,Nz >= 1 cells of dx,dy,dz metres. pbc_a = number of repeats P_a of SetPBC on each side
 * (0 = open boundary). Builds the demagnetising kernel (fp64 on the device, L143) and its
 * real, mirror-symmetric spectrum (L145); cost grows with N and with the PBC repeats.
 * Padded FFT length per open axis: the smallest 2^a 3^b 5^c >= 2N-1 (1 if N == 1), per periodic
 * axis N itself (L509), each <= 8192 (MM_EINVAL beyond, or if a periodic N is not 5-smooth). Open
 * one-layer films of 64..4096 cells per side use twice the next power of two instead (register-FFT
 * kernels; any padded length >= 2N-1 gives the same linear convolution).
 * On success *out owns device memory obtained with cudaMalloc on the current device. */
int mm_create(mm_sim** out, int Nx, int Ny, int Nz, double dx, double dy, double dz, int pbc_x, int pbc_y,
              int pbc_z);

/* As mm_create, with a caller-supplied device allocator (e.g. PyTorch's caching allocator) and
 * CUDA stream (a cudaStream_t; NULL = legacy default stream). dev_alloc returns NULL on failure. */
int mm_create_ex(mm_sim** out, int Nx, int Ny, int Nz, double dx, double dy, double dz, int pbc_x, int pbc_y,
                 int pbc_z, void* (*dev_alloc)(size_t bytes, void* ctx), void (*dev_free)(void* ptr, void* ctx),
                 void* alloc_ctx, void* cuda_stream);

/* Frees the handle and all device memory it owns. NULL is allowed. */
int mm_destroy(mm_sim* sim);

/* Region index of every cell (L43): N bytes [z][y][x]. Default: all 0. */
int mm_set_regions(mm_sim* sim, const uint8_t* regions);

/* Geometry (L53, "B. Geometry", Fig. 2): the shape of the magnet as one byte per cell, [z][y][x], host or device
 * pointer, copied during the call. Non-zero = inside the shape, 0 = outside: such a cell is vacuum whatever its
 * region index says - no magnetisation (m = 0), no exchange coupling to it (a neighbour outside the shape is an
 * open boundary, L196), no torque. The shape does not use up the caller's region indices, but it reserves index
 * 255 of the look-up tables: with a geometry set, mm_set_params accepts at most 255 regions and a region map may
 * not hold index 255 (MM_EINVAL otherwise). NULL removes the geometry. The magnetisation already stored is
 * re-normalised (cells that left the shape become 0; cells that entered it keep 0 until mm_set_m gives them a
 * direction), so mm_set_m usually follows. Errors: MM_EINVAL, MM_ENOMEM, MM_ECUDA. */
int mm_set_geometry(mm_sim* sim, const uint8_t* inside);

/* Material tables and applied field. Rebuilds the device look-up tables (1-D tables per region and
 * the lower-triangular inter-region exchange table, Fig. 1 L31) and invalidates the FSAL slope. */
int mm_set_params(mm_sim* sim, const mm_params* params);

/* Which B_eff terms drive the dynamics (default MM_ALL). */
int mm_set_terms(mm_sim* sim, unsigned term_mask);

/* Implementation switches. MM_OPT_GENERIC_FFT = 1 forces the generic any-size convolution kernels
 * even where a specialised path exists (used by the tests to check the two against each other). */
enum { MM_OPT_GENERIC_FFT = 1,
       MM_OPT_NO_TMA = 2 /* fast 2D x kernels with plain loads/stores instead of TMA tensor copies */,
       MM_OPT_NO_GRAPH = 3 /* launch the kernels of a step one by one instead of replaying a CUDA graph */ };
int mm_set_option(mm_sim* sim, int option, int value);

/* Solver settings (L372-L374). max_err: MaxErr eps0 (default 1e-5); headroom (default 0.8);
 * fix_dt > 0 selects a fixed step (every step accepted), 0 = adaptive; dt_init: first trial step
 * (default 1e-14 s); dt_min/dt_max clip the controller (defaults 1e-18, 1e-9).
 * Pass 0 for any argument to keep its default. */
int mm_set_solver(mm_sim* sim, double max_err, double headroom, double fix_dt, double dt_init, double dt_min,
                  double dt_max);

/* Which embedded Runge-Kutta pair mm_step_rk45 / mm_steps / mm_run advance with (the paper's SetSolver,
 * L805, L853): MM_RK45 = Dormand-Prince 5(4), 7 stages, the default for dynamics (L365); MM_RK23 =
 * Bogacki-Shampine 3(2), 4 stages, used when relaxing (L366, L392). Both are FSAL; the step-size rule
 * uses the exponent 1/5 resp. 1/3. Invalidates the FSAL slope. */
enum { MM_RK45 = 0, MM_RK23 = 1, MM_RK12 = 2 /* Heun 2(1), no FSAL: finite temperature (L367) */ };
int mm_set_solver_kind(mm_sim* sim, int kind);

/* Temperature in kelvin (default 0): inside steps adds the fluctuating field of Eq. 24 (L303-L308),
 * B_therm = eta sqrt(2 mu0 alpha kB T / (Bsat gamma_LL dV dt)), eta standard normal per cell, component and
 * step from a counter-based generator (seed, component, step * N + cell). As the paper requires (L310) a
 * temperature needs the Heun solver and a fixed step: stepping otherwise returns MM_ESTATE.
 * mm_b_eff / mm_torque never include the thermal field. */
int mm_set_temperature(mm_sim* sim, double kelvin, unsigned long long seed);

/* Slonczewski spin-transfer torque (Eq. 28-30) added to every torque evaluation:
 *   tau_SL = beta (eps - alpha eps')/(1+alpha^2) m x (m_P x m) - beta (eps' - alpha eps)/(1+alpha^2) m x m_P,
 *   beta = j_z hbar / (Msat e d), eps = P Lambda^2 / ((Lambda^2+1) + (Lambda^2-1) m.m_P),
 * j_z [A/m^2] through the layer thickness d = Nz dz, polarisation P, Lambda > 0, secondary term eps',
 * fixed-layer direction m_P (normalised by the library; host pointer). As printed beta is a field, so the
 * torque is gamma_LL times the expression (#18). jz = 0 switches the term off. */
int mm_set_slonczewski(mm_sim* sim, double jz, double pol, double lambda, double eps_prime, const double mp[3]);

/* Zhang-Li spin-transfer torque (Eq. 26) added to every torque evaluation:
 *   tau_ZL = 1/(1+alpha^2) [ (1 + xi alpha) m x (m x (u.grad) m) + (xi - alpha) m x (u.grad) m ],
 *   u = mu_B mu0 / (2 e gamma_LL Bsat (1 + xi^2)) j,
 * j [A/m^2] uniform current density (host pointer, 3 doubles), xi the non-adiabaticity. PAPER.md prints both
 * terms identically; the double cross product in the first is DESIGN.md reading #19. Central differences;
 * a missing neighbour at an open boundary is the cell's own m. gamma_LL is the one in force when the
 * torque is evaluated (a later mm_set_params takes effect). j = 0 switches the term off. */
int mm_set_zhang_li(mm_sim* sim, const double j[3], double xi);

/* Interfacial Dzyaloshinskii-Moriya exchange (Eq. 10-17), part of the exchange term MM_EXCH (the paper's
 * E_exch(DM)):  B_DM = (2D/Msat) (dm_z/dx, dm_z/dy, -dm_x/dx - dm_y/dy), central differences (L246), with the boundary
 * conditions of Eq. 11-15: a missing neighbour (outside an open box, or a cell with Msat = 0) is replaced by
 * m + (dm/di)|_dV Delta_i n, dm_z/dx = (D/2A) m_x, dm_x/dx = dm_y/dy = -(D/2A) m_z, dm_z/dy = (D/2A) m_y, others 0;
 * with D != 0 the same virtual neighbours enter the Heisenberg exchange field (L248). D [J/m^2]: n = 1 value for
 * the whole box or n = nregions values (host pointer); D and D/2A are those of the cell's own region (DESIGN.md
 * #20). All zeros (or n = 0) switch the term off. Needs mm_set_params first; energies include Eq. 17. */
int mm_set_dmi(mm_sim* sim, const double* D, int n);

/* Precession term of Eq. 2 on (default) or off: off leaves tau = -gamma alpha/(1+alpha^2) m x (m x B),
 * "so that the effective field points towards decreasing energy" (relax(), L388). */
int mm_set_precession(mm_sim* sim, int on);

/* Reduced magnetisation: 3N floats; normalised to unit length on entry (L85). Cells with
 * Msat = 0 keep m = 0. Invalidates the FSAL slope. mm_get_m copies the current m out. */
int mm_set_m(mm_sim* sim, const float* m);
int mm_get_m(mm_sim* sim, float* m_out);

/* Effective field of the current m for the selected terms, tesla, 3N floats (L108-L113). */
int mm_b_eff(mm_sim* sim, unsigned term_mask, float* B_out);

/* Torque dm/dt of the current m divided by gamma_LL (tesla), all enabled terms (Eq. 2). */
int mm_torque(mm_sim* sim, float* tau_over_gamma_out);

/* One attempted Dormand-Prince step (L365). With info == NULL the step is only enqueued (no
 * synchronisation); otherwise the stream is synchronised and *info filled.
 * MM_ESTATE before mm_set_params + mm_set_m; MM_ENAN if the error estimate is not finite; MM_EDT if a
 * rejected attempt was already at dt_min. After such a failure further steps are no-ops that report the
 * same code until mm_set_solver or mm_set_m clears it; mm_b_eff, mm_torque, mm_energy and mm_max_torque
 * keep working on the (unchanged) magnetisation. */
int mm_step_rk45(mm_sim* sim, mm_step_info* info_or_null);
/* The same call under a solver-neutral name: one attempted step of the selected pair. */
int mm_step(mm_sim* sim, mm_step_info* info_or_null);

/* n attempted steps, enqueued back to back without host synchronisation (the paper's steps(n),
 * L1072, counting rejected attempts too). Synchronises once at the end. */
int mm_steps(mm_sim* sim, int n);

/* Advance time by exactly `duration` seconds (the paper's run(t), L74): the last step is clipped
 * to land on the end time and the controller's suggestion is restored afterwards. The accept /
 * reject decision and the step-size update happen on the device; the host only polls the time.
 * MM_EDT if the step size falls below dt_min; MM_ENAN on a non-finite error estimate. */
int mm_run(mm_sim* sim, double duration);

/* Total energy of the current m for the selected terms, joules: demag Eq. 4 (L125), exchange Eq. 8
 * (L202), anisotropy Eq. 20 / 23 (L278, L297), Zeeman -M.B_ext; fp32 per cell, fp64 sum. */
int mm_energy(mm_sim* sim, unsigned term_mask, double* joules);
/* max over cells of |torque| / gamma_LL [T] of the current m (enabled terms, precession switch as
 * set): the quantity relax() monitors near equilibrium (L388-L390). */
int mm_max_torque(mm_sim* sim, double* tesla);

/* The paper's relax() (L388-L392): with the precession term off and the RK23 pair, advance while the
 * total energy keeps falling, then while the maximum torque keeps falling, decreasing MaxErr each time
 * it stops until MaxErr = 1e-9 (sampled every 3 steps, MaxErr divided by sqrt 2: DESIGN.md #15).
 * Solver kind, precession switch, MaxErr and fixed step are restored; time advances. Host-driven:
 * one scalar crosses to the host per sample. */
int mm_relax(mm_sim* sim);

/* Batched independent simulations (the paper's batch runs and its search over 3000 random starts, L426, L800-L803):
 * `count` handles - typically many small boxes, which alone leave most of the GPU idle (L503) - advance together.
 * Every handle enqueues on its own stream (create them with mm_create, or with distinct streams), so their kernels
 * overlap on the device; the host enqueues a round on all handles before it waits for any. Results are bit for bit
 * those of the same calls made one handle at a time. mm_batch_steps: n attempted steps each; mm_batch_run: advance
 * every handle by `duration`; mm_batch_relax: relax() on every handle. Returns the first error met (all handles are
 * still brought to a consistent state). `sims` is a host array of handles. */
int mm_batch_steps(mm_sim* const* sims, int count, int n);
int mm_batch_run(mm_sim* const* sims, int count, double duration);
int mm_batch_relax(mm_sim* const* sims, int count);

int mm_get_time(mm_sim* sim, double* t);
int mm_set_time(mm_sim* sim, double t);
/* Plain mean of m over all cells (fp64 accumulation), the paper's m.average() (L861). */
int mm_get_avg_m(mm_sim* sim, double avg[3]);
/* The same mean (m.average(), L861) for callers that cannot allocate device memory - code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc. Needs no handle and calls no cudaMalloc, cudaFree
 * or allocating library routine: the per-block partial sums live in one file-scope device array of 196 864 bytes
 * that every GPU loading the library holds until the process exits.
 *   m_dev      DEVICE pointer, 3 * ncells floats, [component][cell] as everywhere in this header (caller-owned, read)
 *   ncells     1 .. MM_NOALLOC_MAX_CELLS; beyond -> MM_EINVAL (the scratch array holds one partial per 8192 cells)
 *   avg_dev    DEVICE pointer, 3 doubles: the mean of each component, fp64 accumulation in an order fixed by ncells
 *              alone (same field -> same bits on any device)
 *   cuda_stream a cudaStream_t (NULL = the default stream); a 4-byte memset and one kernel are enqueued on it, the
 *              call does not synchronise. The device owning the stream and both buffers must be current.
 *   errbuf     optional host buffer of errlen bytes for the text of a failure (may be NULL)
 * The scratch array is shared by EVERY call in the process and keeps the last call's contents (the library clears
 * what must start at zero): calls that overlap on the GPU - different streams without ordering, concurrent graph
 * branches - race on it; order them. The first call on each device looks the array's address up
 * (cudaGetSymbolAddress): make it before starting a capture. */
#define MM_NOALLOC_MAX_CELLS 67108864LL /* 2^26 cells = 8192 x 8192 (a 4096^2 film or a 256^3 cube is 2^24) */
int mm_avg_m_noalloc(const float* m_dev, long long ncells, double* avg_dev, void* cuda_stream, char* errbuf, size_t errlen);
/* Counters: accepted steps, rejected attempts, torque evaluations, peak device bytes owned. */
int mm_get_stats(mm_sim* sim, long* steps, long* rejected, long* evals, size_t* peak_device_bytes);
/* Device bytes the handle owns now and the most it ever owned (the fp64 scratch of the kernel set-up is freed
 * before the vector fields are allocated). The paper's context: about 220 B/cell for 2D RK45 (L533). */
int mm_get_memory(mm_sim* sim, size_t* resident_bytes, size_t* peak_bytes);
/* The CUDA stream all work of this handle is enqueued on (a cudaStream_t). */
int mm_get_stream(mm_sim* sim, void** cuda_stream);
/* Padded FFT sizes chosen for this box (Px, Py, Pz). */
int mm_get_fft_size(mm_sim* sim, int P[3]);
/* Number of kernel launches the library has issued on this handle (for bench.py). */
int mm_get_launch_count(mm_sim* sim, long* launches);

/* Per-kernel timing with CUDA events on the handle's stream (used by bench.py for the roofline
 * line). mm_profile(sim, 1) clears the counters and starts bracketing every launch with a pair of
 * events; mm_profile(sim, 0) stops. mm_profile_read returns, for kernel class `kind`
 * (0 <= kind < 15; MM_EINVAL beyond), its name, the summed duration in ms and the launch count. */
int mm_profile(mm_sim* sim, int enable);
int mm_profile_read(mm_sim* sim, int kind, const char** name, double* total_ms, long* launches);

/* Text of the last failure on a handle; with sim == NULL, of the last failed mm_create on this thread. */
const char* mm_last_error(const mm_sim* sim);
const char* mm_strerror(int code);
const char* mm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MM_B200_H */
