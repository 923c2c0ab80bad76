// implicit_device.cuh — small 3x3 block helpers shared by the assembly kernels (implicit_kernels.cu, assemble_march.cu).
#pragma once
#include "ark_m1_internal.h"

namespace ark {

struct Blk { double a[9]; };

__device__ __forceinline__ void blk_zero(Blk& B) {
#pragma unroll
    for (int k = 0; k < 9; ++k) B.a[k] = 0.0;
}

// Adds w * GL to BL and w * GR to BR for the face `fc` (direction dir) between cells with Jacobians JL, JR.
__device__ __forceinline__ void face_blocks(const Face& fc, int dir, double c2, const Jac& JL, const Jac& JR,
                                            double wL, Blk& BL, double wR, Blk& BR)
{
    const int n = 1 + dir;  // column of the normal flux component
    // energy row
    BL.a[0] += wL * (-fc.alpha * fc.Lam); BL.a[n] += wL * (fc.alpha * fc.ap);
    BR.a[0] += wR * (fc.alpha * fc.Lam);  BR.a[n] += wR * (fc.alpha * fc.am);
    const double* JLx = dir == 0 ? JL.xx : JL.xy; const double* JLy = dir == 0 ? JL.xy : JL.yy;
    const double* JRx = dir == 0 ? JR.xx : JR.xy; const double* JRy = dir == 0 ? JR.xy : JR.yy;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        BL.a[3 + k] += wL * c2 * fc.ap * JLx[k]; BL.a[6 + k] += wL * c2 * fc.ap * JLy[k];
        BR.a[3 + k] += wR * c2 * fc.am * JRx[k]; BR.a[6 + k] += wR * c2 * fc.am * JRy[k];
    }
    BL.a[4] += wL * (-fc.Lam); BL.a[8] += wL * (-fc.Lam);
    BR.a[4] += wR * fc.Lam;    BR.a[8] += wR * fc.Lam;
}

// Inverse of a 3x3 block by cofactors (the blocks are strongly diagonally dominant in practice; a singular
// block yields Inf/NaN which the solver reports as ARK_M1_E_NONFINITE).
__device__ __forceinline__ void inv3(const Blk& B, Blk& I)
{
    const double* a = B.a;
    const double c00 = a[4] * a[8] - a[5] * a[7], c01 = a[5] * a[6] - a[3] * a[8], c02 = a[3] * a[7] - a[4] * a[6];
    const double det = a[0] * c00 + a[1] * c01 + a[2] * c02;
    const double id = rcp_fast(det);
    I.a[0] = c00 * id; I.a[1] = (a[2] * a[7] - a[1] * a[8]) * id; I.a[2] = (a[1] * a[5] - a[2] * a[4]) * id;
    I.a[3] = c01 * id; I.a[4] = (a[0] * a[8] - a[2] * a[6]) * id; I.a[5] = (a[2] * a[3] - a[0] * a[5]) * id;
    I.a[6] = c02 * id; I.a[7] = (a[1] * a[6] - a[0] * a[7]) * id; I.a[8] = (a[0] * a[4] - a[1] * a[3]) * id;
}

// Single-sided form: adds w * G_L (right == false) or w * G_R (right == true) of the face to B, with the Jacobian J of the
// cell on that side.  G_L = [-alpha Lam, alpha a+ e_n ; c^2 a+ J^{n.} - Lam I_F],  G_R = [alpha Lam, alpha a- e_n ; c^2 a- J^{n.} + Lam I_F].
__device__ __forceinline__ void add_G(Blk& B, const Face& fc, int dir, bool right, double w, double c2, const Jac& J)
{
    const int n = 1 + dir;
    const double a = right ? fc.am : fc.ap, sg = right ? 1.0 : -1.0;
    B.a[0] += w * sg * fc.alpha * fc.Lam; B.a[n] += w * fc.alpha * a;
    const double* Jx = dir == 0 ? J.xx : J.xy; const double* Jy = dir == 0 ? J.xy : J.yy;
#pragma unroll
    for (int k = 0; k < 3; ++k) { B.a[3 + k] += w * c2 * a * Jx[k]; B.a[6 + k] += w * c2 * a * Jy[k]; }
    B.a[4] += w * sg * fc.Lam; B.a[8] += w * sg * fc.Lam;
}

}  // namespace ark
