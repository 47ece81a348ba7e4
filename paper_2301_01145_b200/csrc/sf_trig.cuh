// sf_trig.cuh -- the compile-time cosine / sine tables behind the radix-16 and radix-32 butterflies of both kernel
// generations (sf_common.cuh, sf_fast.cuh, sf_fast512.cuh): one definition, usable from any namespace.
#pragma once

namespace sftrig {

// cos / sin of 2 pi i / 16
__host__ __device__ constexpr double cos16(int i)
{
    constexpr double c[16] = { 1.0, 0.92387953251128675613, 0.70710678118654752440, 0.38268343236508977173,
                               0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128675613,
                               -1.0, -0.92387953251128675613, -0.70710678118654752440, -0.38268343236508977173,
                               0.0, 0.38268343236508977173, 0.70710678118654752440, 0.92387953251128675613 };
    return c[i & 15];
}
__host__ __device__ constexpr double sin16(int i) { return cos16(i - 4); }

// cos / sin of 2 pi i / 32
__host__ __device__ constexpr double cos32(int i)
{
    constexpr double c[9] = { 1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                              0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                              0.19509032201612826785, 0.0 };
    i &= 31;
    if (i > 16) i = 32 - i;
    return i <= 8 ? c[i] : -c[16 - i];
}
__host__ __device__ constexpr double sin32(int i) { return cos32(i - 8); }

} // namespace sftrig
