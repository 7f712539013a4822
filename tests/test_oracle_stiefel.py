"""Pins of the oracle's Stiefel step (tangent projection, QR and Newton-Schulz retraction):
invariants, closed forms and library routines.  P:NN = PAPER.md line NN."""
import numpy as np
import pytest

from oracle import mapl_oracle as o


def _orth(rng, d, r):
    q, rr = np.linalg.qr(rng.standard_normal((d, r)))
    return q * np.sign(np.diag(rr))


def _sym(M):
    return 0.5 * (M + M.T)


@pytest.mark.parametrize("d,r", [(20, 4), (33, 7), (16, 16)])
def test_tangent_projection_invariants(d, r):
    """P:115 Eq. 4.  xi is tangent: U^T xi + xi^T U = 0; projection idempotent; matches numpy."""
    rng = np.random.default_rng(d * 100 + r)
    U = _orth(rng, d, r); G = rng.standard_normal((d, r))
    xi = o.tangent(U, G)
    assert np.abs(U.T @ xi + xi.T @ U).max() < 1e-12
    assert np.abs(o.tangent(U, xi) - xi).max() < 1e-12
    assert np.abs(xi - (G - U @ _sym(U.T @ G))).max() < 1e-12
    # G = U K, K symmetric => xi = 0 ;   K skew-symmetric => already tangent => xi = G
    K = _sym(rng.standard_normal((r, r)))
    assert np.abs(o.tangent(U, U @ K)).max() < 1e-12
    W = rng.standard_normal((r, r)); W = W - W.T
    assert np.abs(o.tangent(U, U @ W) - U @ W).max() < 1e-12
    # a NON-symmetric S pins sym(): using S or S^T alone instead of (S+S^T)/2 fails this
    S = U.T @ G
    wrong = G - U @ S
    assert np.abs(xi - wrong).max() > 1e-3


@pytest.mark.parametrize("d,r", [(24, 5), (64, 16), (12, 12)])
def test_qr_retraction(d, r):
    rng = np.random.default_rng(7 * d + r)
    Y = rng.standard_normal((d, r))
    Q, R = o.qr_retract(Y)
    assert np.abs(Q.T @ Q - np.eye(r)).max() < 1e-12
    assert np.abs(np.tril(R, -1)).max() == 0.0 and (np.diag(R) > 0).all()
    assert np.abs(Q @ R - Y).max() < 1e-12
    # library QR with the sign fix
    q, rr = np.linalg.qr(Y); s = np.sign(np.diag(rr))
    assert np.abs(Q - q * s).max() < 1e-11
    # Cholesky closed form: R = chol(Y^T Y)^T, Q = Y R^-1
    Rc = np.linalg.cholesky(Y.T @ Y).T
    assert np.abs(R - Rc).max() < 1e-10
    assert np.abs(Q - Y @ np.linalg.inv(Rc)).max() < 1e-10


def test_qr_retraction_closed_form_on_tangent_step():
    """For tangent xi: Y^T Y = I + lr^2 xi^T xi, so R = chol(I + lr^2 xi^T xi)^T."""
    rng = np.random.default_rng(3)
    d, r, lr = 40, 6, 0.05
    U = _orth(rng, d, r); G = rng.standard_normal((d, r))
    Up, xi = o.stiefel_step(U, G, lr, o.RETRACT_QR)
    Y = U - lr * xi
    assert np.abs(Y.T @ Y - (np.eye(r) + lr * lr * xi.T @ xi)).max() < 1e-12
    Rc = np.linalg.cholesky(np.eye(r) + lr * lr * xi.T @ xi).T
    assert np.abs(Up - Y @ np.linalg.inv(Rc)).max() < 1e-11
    assert np.abs(Up.T @ Up - np.eye(r)).max() < 1e-12


@pytest.mark.parametrize("d,r", [(40, 6), (64, 16)])
def test_newton_schulz_is_polar_factor(d, r):
    """5 cubic NS iterations from Y = U - lr xi reach polar(Y) = Y (I + lr^2 xi^T xi)^(-1/2)
    = U_svd V_svd^T (reading S11)."""
    rng = np.random.default_rng(d + r)
    lr = 0.02
    U = _orth(rng, d, r); G = rng.standard_normal((d, r))
    Up, xi = o.stiefel_step(U, G, lr, o.RETRACT_NS, 5)
    Y = U - lr * xi
    w, V = np.linalg.eigh(np.eye(r) + lr * lr * xi.T @ xi)
    polar = Y @ (V * w ** -0.5) @ V.T
    u, s, vt = np.linalg.svd(Y, full_matrices=False)
    assert s.max() < np.sqrt(3.0)
    assert np.abs(polar - u @ vt).max() < 1e-12
    assert np.abs(Up - polar).max() < 1e-10
    assert np.abs(Up.T @ Up - np.eye(r)).max() < 1e-12


def test_newton_schulz_single_iteration_and_count():
    """one iteration is X (3I - X^T X)/2 exactly; the iteration count is honoured."""
    rng = np.random.default_rng(11)
    Y = _orth(rng, 30, 5) + 0.05 * rng.standard_normal((30, 5))
    X1 = o.newton_schulz(Y, 1)
    assert np.abs(X1 - Y @ (3 * np.eye(5) - Y.T @ Y) / 2).max() < 1e-13
    X2 = o.newton_schulz(Y, 2)
    assert np.abs(X2 - X1 @ (3 * np.eye(5) - X1.T @ X1) / 2).max() < 1e-13
    assert np.abs(o.newton_schulz(Y, 0) - Y).max() == 0.0
    e = [np.linalg.norm(o.newton_schulz(Y, k).T @ o.newton_schulz(Y, k) - np.eye(5)) for k in range(4)]
    assert e[1] < e[0] and e[2] < e[1] ** 1.5      # quadratic convergence


@pytest.mark.parametrize("retr", [o.RETRACT_QR, o.RETRACT_NS])
def test_retractions_first_order_and_fixed_point(retr):
    """Retr(U - t xi) = U - t xi + O(t^2): halving t quarters the error; xi = 0 => U+ = U."""
    rng = np.random.default_rng(5)
    d, r = 36, 5
    U = _orth(rng, d, r); G = rng.standard_normal((d, r))
    errs = []
    for t in (0.02, 0.01, 0.005):
        Up, xi = o.stiefel_step(U, G, t, retr, 5)
        errs.append(np.linalg.norm(Up - (U - t * xi)))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5
    K = _sym(rng.standard_normal((r, r)))
    Up, xi = o.stiefel_step(U, U @ K, 0.1, retr, 5)
    assert np.abs(xi).max() < 1e-12 and np.abs(Up - U).max() < 1e-12


def test_orthonormal_after_every_step_1e12():
    """north_star: U^T U = I after every step, to 1e-12 (oracle)."""
    rng = np.random.default_rng(9)
    d, r = 128, 16
    U = _orth(rng, d, r)
    for retr in (o.RETRACT_QR, o.RETRACT_NS):
        Uc = U.copy()
        for step in range(6):
            G = rng.standard_normal((d, r))
            Uc, _ = o.stiefel_step(Uc, G, 1e-2, retr, 5)
            assert np.linalg.norm(Uc.T @ Uc - np.eye(r)) < 1e-12


# ------------------------------------------------------------------ full SPEL step (Eq. 4-7)

def _scalar_ns(s, iters):
    for _ in range(iters):
        s = 0.5 * s * (3.0 - s * s)
    return s


def test_spel_lmo_direction_matches_svd_with_scalar_iteration():
    """The cubic Newton-Schulz map acts on singular values only: with m_new = P diag(s) Q^T, d = P diag(f(s/||s||)) Q^T where
    f is the scalar iteration s <- s (3 - s^2)/2 applied lmo_iters times (independent computation by numpy SVD)."""
    rng = np.random.default_rng(40)
    d_, r = 40, 6
    U = np.linalg.qr(rng.standard_normal((d_, r)))[0]
    G = rng.standard_normal((d_, r)); m = rng.standard_normal((d_, r))
    beta, lr = 0.9, 0.05
    U2, m2, dirn = o.spel_step(U, G, m, lr, beta, 5, 7)
    xi = o.tangent(U, G)
    assert np.abs(m2 - (beta * m + (1 - beta) * xi)).max() < 1e-13
    P, s, Qt = np.linalg.svd(m2, full_matrices=False)
    f = np.array([_scalar_ns(x, 5) for x in s / np.linalg.norm(s)])
    assert np.abs(dirn - (P * f) @ Qt).max() < 1e-12
    # retraction: orthonormal to 1e-10 (sigma(U - lr d) within [1 - lr, 1 + lr]) and equal to the polar factor
    assert np.linalg.norm(U2.T @ U2 - np.eye(r)) < 1e-10
    Y = U - lr * dirn
    Py, sy, Qyt = np.linalg.svd(Y, full_matrices=False)
    assert np.abs(U2 - Py @ Qyt).max() < 1e-9


def test_spel_special_cases():
    rng = np.random.default_rng(41)
    d_, r = 24, 4
    U = np.linalg.qr(rng.standard_normal((d_, r)))[0]
    G = rng.standard_normal((d_, r))
    # beta = 1: the momentum is untouched, whatever G is
    m = rng.standard_normal((d_, r))
    _, m2, _ = o.spel_step(U, G, m, 0.1, 1.0)
    assert np.array_equal(m2, m)
    # no gradient, no momentum: nothing moves
    U2, m2, dirn = o.spel_step(U, np.zeros_like(G), np.zeros_like(G), 0.1, 0.9)
    assert not dirn.any() and not m2.any() and np.abs(U2 - U).max() < 1e-12
    # momentum with orthonormal columns times a scalar: the direction is f(1/sqrt(r)) times those columns
    W = np.linalg.qr(rng.standard_normal((d_, r)))[0]
    _, _, dirn = o.spel_step(U, np.zeros_like(G), 3.7 * W, 0.1, 1.0, 5, 7)
    assert np.abs(dirn - _scalar_ns(1.0 / np.sqrt(r), 5) * W).max() < 1e-12
