"""CPU ORACLE of the backward pass of the photo term (the transpose of the gather), numpy float64.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this
module. It shares no code with paper_2606_31098_b200/csrc and does not import the C oracle.

What it is ("the refinement is unrolled", supp III-C PAPER.md:427-440): the normal equations of one LM
iteration at pyramid level l are H = sum_j omega_j J_j^T G_j^T G_j J_j, g = sum_j omega_j J_j^T G_j^T r_j over the visible
anchors (Eq.1, Eq.2, Eq.8; SURVEY.md 8(c) EVAL, default GRAD_BILINEAR_EXACT). Given the
gradients G_H = dL/dH (symmetric, dL = <G_H, dH>) and G_g = dL/dg that pilot_oracle's lm_step_adjoint returns, this module
writes out the plain derivative of   S = <G_H, H> + <G_g, g>   with respect to
  * the query feature map F (every tap of every visible anchor),
  * the reference features f^r_j,
  * the pose, as the left perturbation T_cw <- exp(eps^) T_cw, eps = (rho; phi)  (readings A1, A2, A25 of DESIGN.md),
and the query confidence map when there is one, holding the bilinear cell / the visible set fixed (they are piecewise
constant). (Reading A5 holds the weight constant inside the LINEARISATION, i.e. in J; H and g themselves are functions of
the sampled weight w = w_ref wq(u, v), and this is their derivative.)

Per visible anchor, with a, b the bilinear fractions, f00, f10, f01, f11 the taps (C-vectors):
  f  = (1-b)((1-a) f00 + a f10) + b((1-a) f01 + a f11),   gx = (1-b)(f10-f00) + b(f11-f01),   gy = (1-a)(f01-f00) + a(f11-f10)
  r = f - ref,  s = r.r,  x = w s,  omega = w rho'(x)
  A11 = gx.gx, A12 = gx.gy, A22 = gy.gy, b1 = gx.r, b2 = gy.r
  alpha = J G_H J^T (2x2),  beta = J G_g (2),   Q = alpha11 A11 + 2 alpha12 A12 + alpha22 A22 + beta1 b1 + beta2 b2,   S_j = omega Q
  dS/dr  = omega (beta1 gx + beta2 gy) + Q w^2 rho''(x) 2 r
  dS/dgx = omega (2 alpha11 gx + 2 alpha12 gy + beta1 r),   dS/dgy = omega (2 alpha12 gx + 2 alpha22 gy + beta2 r)
  dS/dF_t = wf_t dS/dr + wgx_t dS/dgx + wgy_t dS/dgy  (the tap weights of f, gx, gy),   dS/dref = -dS/dr
  pose, through (u, v):  h = f11 - f01 - f10 + f00;  dS/du = dS/dr.gx + dS/dgy.h,  dS/dv = dS/dr.gy + dS/dgx.h;  J^T (dS/du, dS/dv)
  pose, through J(X, Y, Z):  M = omega (2 A J G_H + b G_g^T) (2x6) = dS/dJ;  sum_pi M_pi dJ_pi/dp . dp/d eps,  dp/d eps = [I | -p^]
  weight:  dS/dw = Q (rho'(x) + x rho''(x));  w = w_ref wq, wq the bilinear sample of the confidence map: dS/dconf_t = dS/dw w_ref wf_t,
           and through (u, v): dS/du += dS/dw w_ref dwq/du (dwq/du = (1-b)(q10-q00) + b(q11-q01)), likewise v
Pins (tests/test_oracle_photo_backward.py): central differences of the C oracle's pilot_oracle_eval (photo term only) with
respect to single map entries, single reference entries and the six pose directions, for the three losses, with and without
confidence weights.
"""
import numpy as np


def loss_d2(kind, x, scale):
    """(rho', rho'') of the robust loss of SURVEY.md 8(c) on x = w ||r||^2."""
    x = np.asarray(x, np.float64)
    if kind == "l2" or not scale > 0:
        return np.ones_like(x), np.zeros_like(x)
    s2 = float(scale) ** 2
    if kind == "huber":
        lin = x > s2
        xs = np.where(lin, x, 1.0)
        return np.where(lin, scale / np.sqrt(xs), 1.0), np.where(lin, -0.5 * scale * xs ** -1.5, 0.0)
    if kind == "cauchy":
        q = 1.0 + x / s2
        return 1.0 / q, -1.0 / (s2 * q * q)
    raise ValueError(kind)


def hat(p):
    return np.array([[0.0, -p[2], p[1]], [p[2], 0.0, -p[0]], [-p[1], p[0], 0.0]])


def photo_backward(feat, ref, points, pose, K, GH, Gg, loss="huber", loss_scale=0.1, z_near=0.1, conf=None):
    """feat [Hh][W][C], ref [N][C], points [N][4] (x, y, z, w_ref), pose [12] = [R_wc | C], K = (fx, fy, cx, cy),
    GH [6][6] symmetric, Gg [6]. Returns (dS/dfeat [Hh][W][C], dS/dref [N][C], dS/d eps [6], S, dS/dconf [Hh][W] or None)."""
    F = np.asarray(feat, np.float64)
    Hh, W, C = F.shape
    ref = np.asarray(ref, np.float64)
    P = np.asarray(points, np.float64)
    T = np.asarray(pose, np.float64).reshape(3, 4)
    R_cw, Cc = T[:, :3].T, T[:, 3]
    fx, fy, cx, cy = [float(k) for k in K]
    GH = np.asarray(GH, np.float64).reshape(6, 6)
    Gg = np.asarray(Gg, np.float64)
    dF, dref, deps, S = np.zeros_like(F), np.zeros_like(ref), np.zeros(6), 0.0
    dconf = None if conf is None else np.zeros((Hh, W))
    for j in range(P.shape[0]):
        p = R_cw @ (P[j, :3] - Cc)
        X, Y, Z = p
        if not Z > z_near:
            continue
        u, v = fx * X / Z + cx, fy * Y / Z + cy
        x0, y0 = int(np.floor(u)), int(np.floor(v))
        if x0 < 0 or y0 < 0 or x0 + 1 > W - 1 or y0 + 1 > Hh - 1:
            continue
        a, b = u - x0, v - y0
        f00, f10, f01, f11 = F[y0, x0], F[y0, x0 + 1], F[y0 + 1, x0], F[y0 + 1, x0 + 1]
        f = (1 - b) * ((1 - a) * f00 + a * f10) + b * ((1 - a) * f01 + a * f11)
        gx = (1 - b) * (f10 - f00) + b * (f11 - f01)
        gy = (1 - a) * (f01 - f00) + a * (f11 - f10)
        w = P[j, 3]
        wq_u = wq_v = 0.0
        if conf is not None:
            q = np.asarray(conf, np.float64)
            q00, q10, q01, q11 = q[y0, x0], q[y0, x0 + 1], q[y0 + 1, x0], q[y0 + 1, x0 + 1]
            w = w * ((1 - b) * ((1 - a) * q00 + a * q10) + b * ((1 - a) * q01 + a * q11))
            wq_u = (1 - b) * (q10 - q00) + b * (q11 - q01)
            wq_v = (1 - a) * (q01 - q00) + a * (q11 - q10)
        r = f - ref[j]
        x = w * (r @ r)
        d1, d2 = loss_d2(loss, x, loss_scale)
        om = w * float(d1)
        J = np.array([[fx / Z, 0, -fx * X / Z ** 2, -fx * X * Y / Z ** 2, fx * (1 + X * X / Z ** 2), -fx * Y / Z],
                      [0, fy / Z, -fy * Y / Z ** 2, -fy * (1 + Y * Y / Z ** 2), fy * X * Y / Z ** 2, fy * X / Z]])
        A = np.array([[gx @ gx, gx @ gy], [gx @ gy, gy @ gy]])
        bb = np.array([gx @ r, gy @ r])
        al, be = J @ GH @ J.T, J @ Gg
        Q = al[0, 0] * A[0, 0] + 2 * al[0, 1] * A[0, 1] + al[1, 1] * A[1, 1] + be @ bb
        S += om * Q
        Sr = om * (be[0] * gx + be[1] * gy) + Q * w * w * float(d2) * 2.0 * r
        Sgx = om * (2 * al[0, 0] * gx + 2 * al[0, 1] * gy + be[0] * r)
        Sgy = om * (2 * al[0, 1] * gx + 2 * al[1, 1] * gy + be[1] * r)
        wf = [(1 - a) * (1 - b), a * (1 - b), (1 - a) * b, a * b]
        wgx = [-(1 - b), (1 - b), -b, b]
        wgy = [-(1 - a), -a, (1 - a), a]
        for t, (yy, xx) in enumerate([(y0, x0), (y0, x0 + 1), (y0 + 1, x0), (y0 + 1, x0 + 1)]):
            dF[yy, xx] += wf[t] * Sr + wgx[t] * Sgx + wgy[t] * Sgy
        dref[j] -= Sr
        # pose through (u, v)
        h = f11 - f01 - f10 + f00
        Su, Sv = Sr @ gx + Sgy @ h, Sr @ gy + Sgx @ h
        if conf is not None:
            Sw = Q * (float(d1) + x * float(d2))
            Su += Sw * P[j, 3] * wq_u
            Sv += Sw * P[j, 3] * wq_v
            for t, (yy, xx) in enumerate([(y0, x0), (y0, x0 + 1), (y0 + 1, x0), (y0 + 1, x0 + 1)]):
                dconf[yy, xx] += Sw * P[j, 3] * wf[t]
        deps += J.T @ np.array([Su, Sv])
        # pose through J(X, Y, Z)
        M = om * (2 * A @ J @ GH + np.outer(bb, Gg))
        iz = 1.0 / Z
        dJ_dX = np.array([[0, 0, -fx * iz ** 2, -fx * Y * iz ** 2, 2 * fx * X * iz ** 2, 0],
                          [0, 0, 0, 0, fy * Y * iz ** 2, fy * iz]])
        dJ_dY = np.array([[0, 0, 0, -fx * X * iz ** 2, 0, -fx * iz],
                          [0, 0, -fy * iz ** 2, -2 * fy * Y * iz ** 2, fy * X * iz ** 2, 0]])
        dJ_dZ = np.array([[-fx * iz ** 2, 0, 2 * fx * X * iz ** 3, 2 * fx * X * Y * iz ** 3, -2 * fx * X * X * iz ** 3, fx * Y * iz ** 2],
                          [0, -fy * iz ** 2, 2 * fy * Y * iz ** 3, 2 * fy * Y * Y * iz ** 3, -2 * fy * X * Y * iz ** 3, -fy * X * iz ** 2]])
        Sp = np.array([np.sum(M * dJ_dX), np.sum(M * dJ_dY), np.sum(M * dJ_dZ)])
        deps += np.concatenate([np.eye(3), -hat(p)], 1).T @ Sp
    return dF, dref, deps, S, dconf
