// sh_math.cuh — real spherical harmonics of degree <= 3 and their R^3 polynomial gradients
// (eq.(5); basis convention: DESIGN.md reading R15, j = l^2+l+m, Condon-Shortley sign kept).
#pragma once

namespace nasg {

// Y_J(x,y,z) and its R^3 polynomial gradient, J compile-time so the unrolled loop keeps only the
// terms of one basis function live.
template <int J>
__device__ __forceinline__ void sh_term(float x, float y, float z, float &Y, float &gx, float &gy, float &gz)
{
    constexpr float C0 = 0.28209479177387814f, C1 = 0.4886025119029199f;
    constexpr float C2A = 1.0925484305920792f, C2B = 0.31539156525252005f, C2C = 0.5462742152960396f;
    constexpr float C3A = 0.5900435899266435f, C3B = 2.890611442640554f, C3C = 0.4570457994644658f,
                    C3D = 0.3731763325901154f, C3E = 1.445305721320277f;
    const float xx = x * x, yy = y * y, zz = z * z;
    if constexpr (J == 0) { Y = C0; gx = 0.f; gy = 0.f; gz = 0.f; }
    else if constexpr (J == 1) { Y = -C1 * y; gx = 0.f; gy = -C1; gz = 0.f; }
    else if constexpr (J == 2) { Y = C1 * z; gx = 0.f; gy = 0.f; gz = C1; }
    else if constexpr (J == 3) { Y = -C1 * x; gx = -C1; gy = 0.f; gz = 0.f; }
    else if constexpr (J == 4) { Y = C2A * x * y; gx = C2A * y; gy = C2A * x; gz = 0.f; }
    else if constexpr (J == 5) { Y = -C2A * y * z; gx = 0.f; gy = -C2A * z; gz = -C2A * y; }
    else if constexpr (J == 6) { Y = C2B * (2.f * zz - xx - yy); gx = -2.f * C2B * x; gy = -2.f * C2B * y; gz = 4.f * C2B * z; }
    else if constexpr (J == 7) { Y = -C2A * x * z; gx = -C2A * z; gy = 0.f; gz = -C2A * x; }
    else if constexpr (J == 8) { Y = C2C * (xx - yy); gx = 2.f * C2C * x; gy = -2.f * C2C * y; gz = 0.f; }
    else if constexpr (J == 9) { Y = -C3A * y * (3.f * xx - yy); gx = -6.f * C3A * x * y; gy = -3.f * C3A * (xx - yy); gz = 0.f; }
    else if constexpr (J == 10) { Y = C3B * x * y * z; gx = C3B * y * z; gy = C3B * x * z; gz = C3B * x * y; }
    else if constexpr (J == 11) { Y = -C3C * y * (4.f * zz - xx - yy); gx = 2.f * C3C * x * y; gy = -C3C * (4.f * zz - xx - 3.f * yy); gz = -8.f * C3C * y * z; }
    else if constexpr (J == 12) { Y = C3D * z * (2.f * zz - 3.f * xx - 3.f * yy); gx = -6.f * C3D * x * z; gy = -6.f * C3D * y * z; gz = 3.f * C3D * (2.f * zz - xx - yy); }
    else if constexpr (J == 13) { Y = -C3C * x * (4.f * zz - xx - yy); gx = -C3C * (4.f * zz - 3.f * xx - yy); gy = 2.f * C3C * x * y; gz = -8.f * C3C * x * z; }
    else if constexpr (J == 14) { Y = C3E * z * (xx - yy); gx = 2.f * C3E * x * z; gy = -2.f * C3E * y * z; gz = C3E * (xx - yy); }
    else { Y = -C3A * x * (xx - 3.f * yy); gx = -3.f * C3A * (xx - yy); gy = 6.f * C3A * x * y; gz = 0.f; }
}

} // namespace nasg
