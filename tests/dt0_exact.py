"""Extended-precision anchor for the fluid increment dT^0_alpha ("What's weak" 1).

Test code only.  The coupling of one cell (Eq.33b, 38, 40, 42, 48-50) is evaluated here in numpy's long double
(64-bit mantissa on x86-64: unit roundoff 5.4e-20, 2048 times finer than FP64's) from the SAME FP64 inputs the oracle and the CUDA
path receive: the oracle's geometry records, the fluid state, the opacities and the pre-coupling intensities I*.  With N <= 400
angles its own rounding (~ N 5e-20 |R^0_0|) is three orders of magnitude below what is being measured, so it stands in for the
exact-arithmetic result.  Both implementations are then measured against it in units of eps |R^0_0| (eps = 2^-53):

    k = |dT^0_alpha (implementation) - dT^0_alpha (long double)| / (2^-53 |R^0_0|)

which is what parity_util.dt0_floor claims to bound (k <= 2 sqrt(N) per side, so that two correct implementations differ by at most
4 sqrt(N) eps |R^0_0|).  Neither the oracle nor the CUDA path is imported here; the arithmetic below is the paper's, retyped.
"""
import numpy as np

LD = np.longdouble
PI = LD(np.pi) + LD(1.2246467991473532e-16)  # pi to long double: the FP64 value plus its residual


def assert_long_double_is_extended():
    assert np.finfo(LD).nmant >= 63, "this platform's long double is not the x87 extended format: the anchor would prove nothing"


def doppler_factors(cell, nhat, fluid):
    """n^0bar = u^0hat - u^ahat n^ahat [C][N] in long double, from the oracle's cell records and the fluid's normal-frame velocity"""
    cell = cell.astype(LD); nh = nhat.astype(LD); up = fluid[2:5].astype(LD).T
    alpha = cell[:, 0]; L = cell[:, 17:33].reshape(-1, 4, 4); beta = cell[:, 63:66]; gm = cell[:, 66:72]
    gam = np.stack([np.stack([gm[:, 0], gm[:, 1], gm[:, 2]], -1), np.stack([gm[:, 1], gm[:, 3], gm[:, 4]], -1), np.stack([gm[:, 2], gm[:, 4], gm[:, 5]], -1)], 1)
    W = np.sqrt(1 + np.einsum("cpq,cp,cq->c", gam, up, up))
    ucon = np.concatenate([(W / alpha)[:, None], up - beta * (W / alpha)[:, None]], 1)
    uh = np.einsum("cba,cb->ca", L, ucon) * np.array([-1, 1, 1, 1], dtype=LD)
    return uh[:, :1] - uh[:, 1:] @ nh.T


def coupling_increment(cell, nhat, domega, fluid, opac, Istar, dt, gamma_gas, a_rad, renorm=True):
    """cell: [C][72] oracle records (alpha, e[mu][ahat], L[mu][ahat], S, beta, gamma_ab); nhat [N][3]; domega [N]; fluid [5][C] = rho, T,
    u^1', u^2', u^3'; opac [3][C]; Istar [C][N].  Returns (dT0 [4][C], T_plus [C], ok [C] bool, R00 [C]) as long doubles / bools."""
    cell = cell.astype(LD); nh = nhat.astype(LD); dOm = domega.astype(LD); I = Istar.astype(LD)
    rho, Tm, up = fluid[0].astype(LD), fluid[1].astype(LD), fluid[2:5].astype(LD).T      # up: [C][3]
    aP, aEa, aS = (opac[q].astype(LD) for q in range(3))
    dt = LD(dt); gamma_gas = LD(gamma_gas); a_rad = LD(a_rad)
    alpha = cell[:, 0]
    e = cell[:, 1:17].reshape(-1, 4, 4); L = cell[:, 17:33].reshape(-1, 4, 4)
    beta = cell[:, 63:66]; gm = cell[:, 66:72]
    gam = np.stack([np.stack([gm[:, 0], gm[:, 1], gm[:, 2]], -1), np.stack([gm[:, 1], gm[:, 3], gm[:, 4]], -1), np.stack([gm[:, 2], gm[:, 4], gm[:, 5]], -1)], 1)
    # R10: Lorentz factor in the normal frame, coordinate four-velocity (inverse of Eq.7)
    W = np.sqrt(1 + np.einsum("cpq,cp,cq->c", gam, up, up))
    ucon = np.concatenate([(W / alpha)[:, None], up - beta * (W / alpha)[:, None]], 1)
    # u^ahat = eta^{ahat ahat} L[beta][ahat] u^beta (Eq.8b, 9)
    uh = np.einsum("cba,cb->ca", L, ucon) * np.array([-1, 1, 1, 1], dtype=LD)
    n4 = np.concatenate([np.ones((nh.shape[0], 1), dtype=LD), nh], 1)                     # (1, nhat) [N][4]
    n0bar = uh[:, :1] - uh[:, 1:] @ nh.T                                                  # P:L309  [C][N]
    dOmb = dOm[None, :] / n0bar ** 2                                                      # R11
    Ibm = n0bar ** 4 * I
    if renorm:
        dOmb = 4 * PI * dOmb / dOmb.sum(1, keepdims=True)                                 # R12
    aE = aEa + aS                                                                          # Eq.33b
    nup0 = e[:, 0, :] @ n4[0]                                                              # n^0 (the same for every angle: e^0_ahat = 0)
    dn = nup0[:, None] + n0bar * (aE * dt)[:, None]
    A1 = ((nup0[:, None] / dn) * Ibm * dOmb).sum(1)                                        # Eq.42a
    A2 = ((n0bar / dn) * dOmb).sum(1) * dt / (4 * PI)                                      # Eq.42b
    Em = (Ibm * dOmb).sum(1)                                                               # Eq.38
    Cv = rho / (gamma_gas - 1)
    B4 = A2 * aP * a_rad; B1 = Cv * (1 - A2 * aS); B0 = A1 - (1 - A2 * aS) * Em - B1 * Tm  # Eq.50
    ok = (B0 < 0) & (B1 > 0) & (B4 >= 0)
    # Eq.49: the positive root of B4 T^4 + B1 T + B0, Newton from the upper bound (convex, increasing: monotone from the right)
    with np.errstate(all="ignore"):
        T = np.where(ok, np.minimum(-B0 / B1, np.where(B4 > 0, np.sqrt(np.sqrt(-B0 / np.where(B4 > 0, B4, 1))), np.inf)), Tm)
        for _ in range(200):
            g = B4 * T ** 4 + B1 * T + B0
            step = np.where(ok, g / (4 * B4 * T ** 3 + B1), 0)
            T = T - step
            if np.all(np.abs(step) <= LD(1e-19) * np.abs(T)):
                break
    Ep = Em - Cv * (T - Tm)                                                                # Eq.48
    src = aP * a_rad * T ** 4 + aS * Ep
    Ibp = (nup0[:, None] * Ibm + n0bar * (dt / (4 * PI)) * src[:, None]) / dn              # Eq.40
    Inew = Ibp / n0bar ** 4
    nlow = np.einsum("cma,na->cmn", L, n4)                                                 # n_alpha = L[alpha][ahat] n^ahat  [C][4][N]
    wgt = nup0[:, None, None] * nlow * dOm[None, None, :]
    dT0 = -(wgt * (Inew - I)[:, None, :]).sum(2)
    dT0 = np.where(ok[:, None], dT0, 0)
    R00 = np.abs((wgt[:, 0, :] * I).sum(1))
    return dT0.T, np.where(ok, T, Tm), ok, R00
