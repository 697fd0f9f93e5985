// common.cuh - shared declarations of the CUDA path (sm_100a). Not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/mm.h"

#define MM_THERMAL 16u   /* internal term bit: thermal field of the current step (never part of MM_ALL) */
#define MM_DMI_ON 32u    /* internal term bit: a Dzyaloshinskii-Moriya strength is set (exchange part takes the boundary-condition path) */
#define MM_TRI_ENTRIES (MM_MAX_REGIONS * (MM_MAX_REGIONS + 1) / 2)

// ---- buffer roles: every kernel fetches its array pointers from DevState::ptr[role], so that the
// accept/reject decision (taken on the device) can swap roles without a host round trip.
enum Role { R_M = 0, R_MNEW, R_Y, R_K0, R_K1, R_K2, R_K3, R_K4, R_K5, R_K6, R_B, R_Y2, R_COUNT };   // R_Y / R_Y2: stage inputs, alternating

struct DevState {
  float* ptr[R_COUNT];
  double t;          // simulation time [s]
  double dt;         // controller's current step suggestion [s]
  double h;          // step being attempted [s]
  double t_end;      // run target (used when run_mode)
  double keep_dt;    // suggestion saved while a clipped step is attempted
  double run_duration;
  double max_err, headroom, fix_dt, dt_min, dt_max, gamma;
  float hg;          // gamma * h as float (torque slopes are kept in tesla)
  unsigned err_bits; // float bits of max || sum_j e_j k_j ||  (atomicMax; non-negative floats order as uints)
  float last_err;
  int nstage;        // stages of the embedded pair: 7 (Dormand-Prince), 4 (Bogacki-Shampine), 2 (Heun)
  int nevals;        // torque evaluations per attempted step: 6, 3, 2
  double temperature;            // kelvin; > 0 adds the thermal field of Eq. 24 inside steps
  unsigned long long seed;       // of the counter-based generator behind eta
  float therm_scale;             // sqrt(T / h) of the current attempt
  double expo;       // exponent of the step-size rule: 1/5 or 1/3
  int run_mode;      // 1: stop at t_end
  int clipped;       // current attempt was clipped to land on t_end
  int skip;          // 1: t_end reached (or failure) -> every kernel of the step returns at once
  int have_k1;       // FSAL slope valid
  int last_accepted;
  int status;        // MM_OK, MM_ENAN, MM_EDT
  long long steps, rejected, evals;
};

// ---- per-region look-up tables (Fig. 1), fp32 on the device
struct Luts {
  float Bsat[MM_MAX_REGIONS];   // mu0 * Msat [T]
  float alpha[MM_MAX_REGIONS];
  float live[MM_MAX_REGIONS];   // 1 if Msat > 0 else 0
  float therm[MM_MAX_REGIONS];  // sqrt(2 mu0 alpha kB / (Bsat gamma dV)) [T sqrt(s/K)]   (Eq. 24 without T and dt)
  float ku1[MM_MAX_REGIONS];    // 2 Ku1 / Msat [T]           (Eq. 18)
  float ku2[MM_MAX_REGIONS];    // 4 Ku2 / Msat [T]
  float u[3][MM_MAX_REGIONS];
  float kc1[MM_MAX_REGIONS];    // -2 Kc1 / Msat [T]          (Eq. 21)
  float kc2[MM_MAX_REGIONS];    // -2 Kc2 / Msat
  float kc3[MM_MAX_REGIONS];    // -4 Kc3 / Msat
  float c1[3][MM_MAX_REGIONS], c2[3][MM_MAX_REGIONS], c3[3][MM_MAX_REGIONS];
  float bext[4];
  int nregions;
  int has_uniaxial, has_cubic;
  float dmi[MM_MAX_REGIONS];    // 2 D / Msat [T m]            (Eq. 10)
  float dmi_bc[MM_MAX_REGIONS]; // D / (2 Aex) [1/m]: boundary derivative of Eq. 11-13
  float exch[MM_TRI_ENTRIES];   // 2 * L[i,j] [T m^2], lower triangular i(i+1)/2 + j, i >= j (Eq. 9)
};

// ---- FFT plan of one axis: Stockham autosort passes over radices {8,4,2,3,5}
#define MM_MAX_PASSES 16
struct AxisPlan {
  int N;        // physical cells along the axis
  int P;        // padded transform length (N if periodic, 1 if N == 1)
  int npass;
  int radix[MM_MAX_PASSES];
};

struct Geometry {
  int Nx, Ny, Nz;
  int Px, Py, Pz;
  int Cx;        // Px/2 + 1 stored kx
  int pitch;     // row pitch of the spectrum in complex elements (>= Cx)
  int Hy, Hz;    // Py/2 + 1, Pz/2 + 1: extent of the symmetric kernel spectrum
  int pbc[3];
  float inv_dx2, inv_dy2, inv_dz2;
  float dx, dy;  // cell edges [m] (central differences and boundary conditions of the DM term)
  long long N;   // cells
};

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
