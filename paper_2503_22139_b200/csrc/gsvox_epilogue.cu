// gsvox_epilogue.cu — step a5: per-Gaussian chain rule (DESIGN.md section 2,
// "Backward").  Reads the u-frame moment sums a4 accumulated, maps them back to d = x - p
// through the unit-triangular L of M = L D L^T, converts to world units and applies
//   dL/dp = M S1,  D_M = -1/2 S2,  dL/ds_k = -2 (R^T D_M R)_kk / s_k^3,
//   D_R = 2 D_M R diag(1/s^2),  dL/dq^ = <dR/dq^, D_R>,  dL/dq = (dL/dq^ - q^ (q^.dL/dq^)) / |q|.
#include "gsvox_internal.cuh"

namespace gsvox {

// ------------------------------------------------------------------------------------------
// a5: chain rule, one thread per Gaussian, fp64 (negligible cost; keeps the rounding of the
// kernel's fp32 sums the only fp32 error in the gradients).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 3)
k_epilogue(const GsAux* __restrict__ aux, const GsRec* __restrict__ rec, const float* __restrict__ acc, int astride, int n, int C,
           GridDev gd, const DevStatus* __restrict__ status,
           float* __restrict__ gw, float* __restrict__ gp, float* __restrict__ gs, float* __restrict__ gq)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const GsAux a = aux[i];
    const bool dead = (a.valid == 0u) || (status->overflow != 0u);
    const float* m = acc + (size_t)i * astride;
    for (int c = 0; c < C; ++c) gw[(size_t)i * C + c] = dead ? 0.f : m[9 + c];
    if (dead) {
        for (int k = 0; k < 3; ++k) { gp[3 * i + k] = 0.f; gs[3 * i + k] = 0.f; }
        for (int k = 0; k < 4; ++k) gq[4 * i + k] = 0.f;
        return;
    }
    const double h[3] = { gd.spacing[0], gd.spacing[1], gd.spacing[2] };
    // u-frame -> index-frame moments: d = T u, T = L^-T (unit upper triangular), with the
    // fp32 l's the kernel used; then world units: S1 = H T mu, S2 = H T B T^T H
    const GsRec rc = rec[i];
    const double l01 = -(double)rc.nl01, l02 = -(double)rc.nl02, l12 = (double)rc.l12;
    const double T[9] = { 1.0, -l01, l01 * l12 - l02,   0.0, 1.0, -l12,   0.0, 0.0, 1.0 };
    const double mu[3] = { m[0], m[1], m[2] };
    const double B[9] = { m[3], m[4], m[5],   m[4], m[6], m[7],   m[5], m[7], m[8] };
    double S1[3], TB[9], S2[9];
    for (int a2 = 0; a2 < 3; ++a2) {
        S1[a2] = (T[3 * a2] * mu[0] + T[3 * a2 + 1] * mu[1] + T[3 * a2 + 2] * mu[2]) * h[a2];
        for (int k = 0; k < 3; ++k)
            TB[3 * a2 + k] = T[3 * a2] * B[k] + T[3 * a2 + 1] * B[3 + k] + T[3 * a2 + 2] * B[6 + k];
    }
    for (int a2 = 0; a2 < 3; ++a2)
        for (int k = 0; k < 3; ++k)
            S2[3 * a2 + k] = (TB[3 * a2] * T[3 * k] + TB[3 * a2 + 1] * T[3 * k + 1] + TB[3 * a2 + 2] * T[3 * k + 2])
                             * h[a2] * h[k];
    double q[4] = { a.q[0], a.q[1], a.q[2], a.q[3] }, s[3] = { a.s[0], a.s[1], a.s[2] };
    double qn = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    double r = q[0] / qn, x = q[1] / qn, y = q[2] / qn, z = q[3] / qn;
    double R[9] = { 1 - 2 * (y * y + z * z), 2 * (x * y - r * z), 2 * (x * z + r * y),
                    2 * (x * y + r * z), 1 - 2 * (x * x + z * z), 2 * (y * z - r * x),
                    2 * (x * z - r * y), 2 * (y * z + r * x), 1 - 2 * (x * x + y * y) };
    double is2[3] = { 1.0 / (s[0] * s[0]), 1.0 / (s[1] * s[1]), 1.0 / (s[2] * s[2]) };
    // dL/dp = M S1, M = R diag(1/s^2) R^T : t = R^T S1, scaled, rotated back
    double t[3];
    for (int k = 0; k < 3; ++k) t[k] = (R[k] * S1[0] + R[3 + k] * S1[1] + R[6 + k] * S1[2]) * is2[k];
    for (int a2 = 0; a2 < 3; ++a2) gp[3 * i + a2] = (float)(R[3 * a2] * t[0] + R[3 * a2 + 1] * t[1] + R[3 * a2 + 2] * t[2]);
    // D_M = -1/2 S2;  P = D_M R
    double P[9];
    for (int a2 = 0; a2 < 3; ++a2)
        for (int k = 0; k < 3; ++k)
            P[3 * a2 + k] = -0.5 * (S2[3 * a2] * R[k] + S2[3 * a2 + 1] * R[3 + k] + S2[3 * a2 + 2] * R[6 + k]);
    // dL/ds_k = -2 (R^T D_M R)_kk / s_k^3
    for (int k = 0; k < 3; ++k) {
        double d = R[k] * P[k] + R[3 + k] * P[3 + k] + R[6 + k] * P[6 + k];
        gs[3 * i + k] = (float)(-2.0 * d * is2[k] / s[k]);
    }
    // D_R = 2 D_M R diag(1/s^2);  dL/dq^_j = <dR/dq^_j, D_R>
    double DR[9];
    for (int a2 = 0; a2 < 3; ++a2) for (int k = 0; k < 3; ++k) DR[3 * a2 + k] = 2.0 * P[3 * a2 + k] * is2[k];
    double gh[4];
    gh[0] = 2 * (-z * DR[1] + y * DR[2] + z * DR[3] - x * DR[5] - y * DR[6] + x * DR[7]);
    gh[1] = 2 * (y * DR[1] + z * DR[2] + y * DR[3] - 2 * x * DR[4] - r * DR[5] + z * DR[6] + r * DR[7] - 2 * x * DR[8]);
    gh[2] = 2 * (-2 * y * DR[0] + x * DR[1] + r * DR[2] + x * DR[3] + z * DR[5] - r * DR[6] + z * DR[7] - 2 * y * DR[8]);
    gh[3] = 2 * (-2 * z * DR[0] - r * DR[1] + x * DR[2] + r * DR[3] - 2 * z * DR[4] + y * DR[5] + x * DR[6] + y * DR[7]);
    double qh[4] = { r, x, y, z };
    double dot = qh[0] * gh[0] + qh[1] * gh[1] + qh[2] * gh[2] + qh[3] * gh[3];
    for (int k = 0; k < 4; ++k) gq[4 * i + k] = (float)((gh[k] - qh[k] * dot) / qn);
}


int launch_epilogue(gsvox_plan* p, int channels, float* gw, float* gp, float* gs, float* gq, cudaStream_t st)
{
    LaunchScope ls(p, GSVOX_K_EPILOGUE, st);
    int blocks = (int)((p->n + 255) / 256);
    k_epilogue<<<blocks, 256, 0, st>>>(p->aux, p->rec, p->acc, acc_stride(channels), (int)p->n, channels, p->gd,
                                       p->status, gw, gp, gs, gq);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

}  // namespace gsvox
