// md.cu -- device-resident molecular dynamics around the energy/force path: velocity Verlet
// with a Nose-Hoover thermostat (the paper runs its potentials in NVT MD at 300 K; MD driver
// of section 4.2). The integrator is the one stated in DESIGN.md section 2, reading B-8:
//     thermostat half step,  v += dt/2 a,  x += dt v,  a = F(x) / m,  v += dt/2 a,  thermostat half step
//     thermostat: dv/dt = -vxi v,  dvxi/dt = (2 KE - g kB T) / Q,  dxi/dt = vxi,  Q = g kB T tau^2,  g = 3 N
//     half step h = dt/2:  vxi += h/2 G;  v *= exp(-h vxi);  xi += h vxi;  vxi += h/2 G   (G from the current KE)
// Positions, velocities, forces and the thermostat variables live on the device for the whole run. The velocity
// scaling of a thermostat half step is never a pass of its own: the kinetic energy after a scaling is known
// analytically (KE s^2), so the half step that closes step k and the one that opens step k+1 are one single-thread
// update (k_nh_update) fed by ONE kinetic-energy reduction per step (fused into the second half kick), and the
// product of their two scale factors is applied inside the next kick+drift kernel.
#include "common.cuh"

namespace {

constexpr int MD_TPB = 256;

// state[0] = xi, [1] = vxi, [2] = scale to apply before the next kick, [3] = 2 KE (eV) of the velocities as they
// will be after that scaling, [4] = scale still to be applied at the end of the run
__global__ void __launch_bounds__(MD_TPB) k_md_kick(int64_t N, double *__restrict__ pos, double *__restrict__ vel,
                                                   const double *__restrict__ F, const double *__restrict__ inv_mass,
                                                   double dt, double acc_unit, int drift, const double *__restrict__ state,
                                                   double *__restrict__ ke_partial) {
    __shared__ double red[MD_TPB];
    const int64_t i = (int64_t)blockIdx.x * MD_TPB + threadIdx.x;
    const double pre = (state && drift) ? state[2] : 1.0;
    double mv2 = 0.0;
    if (i < N) {
        const double im = inv_mass[i], s = 0.5 * dt * acc_unit * im;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double v = __dmul_rn(vel[3 * i + d], pre) + s * F[3 * i + d];
            vel[3 * i + d] = v;
            if (drift) pos[3 * i + d] += dt * v;
            mv2 += v * v;
        }
        mv2 /= im;
    }
    if (!ke_partial) return;
    red[threadIdx.x] = mv2;
    __syncthreads();
    for (int s = MD_TPB / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) ke_partial[blockIdx.x] = red[0];
}

// sum of the block partials (fixed order), then the thermostat algebra; one block
//   mode 0: first half step of the run (opens step 1);  1: closes a step and opens the next;  2: closes the last step
__global__ void __launch_bounds__(MD_TPB) k_nh_update(int nb, const double *__restrict__ ke_partial, double *__restrict__ state,
                                                     double h, double g_kT, double Q, double acc_unit, int mode, int nvt) {
    __shared__ double red[MD_TPB];
    double s = 0.0;
    for (int k = threadIdx.x; k < nb; k += MD_TPB) s += ke_partial[k];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int st = MD_TPB / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) red[threadIdx.x] += red[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    double ke2 = red[0] / acc_unit, xi = state[0], vxi = state[1], scale = 1.0;
    if (nvt) {
        const int halves = mode == 1 ? 2 : 1;
        for (int k = 0; k < halves; ++k) {
            vxi += 0.5 * h * (ke2 - g_kT) / Q;
            const double sc = exp(-h * vxi);
            scale *= sc;
            ke2 *= sc * sc;
            xi += h * vxi;
            vxi += 0.5 * h * (ke2 - g_kT) / Q;
        }
    }
    state[0] = xi; state[1] = vxi; state[3] = ke2;
    if (mode == 2) { state[2] = 1.0; state[4] = scale; }
    else { state[2] = scale; state[4] = 1.0; }
}

__global__ void __launch_bounds__(MD_TPB) k_md_scale(int64_t n3, double *__restrict__ vel, const double *__restrict__ state) {
    const int64_t i = (int64_t)blockIdx.x * MD_TPB + threadIdx.x;
    if (i < n3) vel[i] = __dmul_rn(vel[i], state[4]);
}

} // namespace

int md_blocks(int64_t N) { return (int)div_up(N > 0 ? N : 1, MD_TPB); }

void launch_md_kick(const LaunchCtx &ctx, int64_t N, double *pos, double *vel, const double *F, const double *inv_mass,
                    double dt, double acc_unit, int drift, const double *state, double *ke_partial) {
    LAUNCH(ctx, k_md_kick, md_blocks(N), MD_TPB, 0, N, pos, vel, F, inv_mass, dt, acc_unit, drift, state, ke_partial);
}
void launch_nh_update(const LaunchCtx &ctx, int64_t N, const double *ke_partial, double *state, double h, double g_kT,
                      double Q, double acc_unit, int mode, int nvt) {
    LAUNCH(ctx, k_nh_update, 1, MD_TPB, 0, md_blocks(N), ke_partial, state, h, g_kT, Q, acc_unit, mode, nvt);
}
void launch_md_scale(const LaunchCtx &ctx, int64_t N, double *vel, const double *state) {
    if (N > 0) LAUNCH(ctx, k_md_scale, div_up(3 * N, MD_TPB), MD_TPB, 0, 3 * N, vel, state);
}
