"""Paper-style kernel tables: the weighted least-squares split of a radial kernel K_l into a truncated l-space
part and a truncated real-space part (Eq. 1-5), for a flat input spectrum.

This is INPUT GENERATION for the convolution path (CPU pre-processing in the paper): it holds
none of the convolution's arithmetic and is used by tests / examples only.  numpy only.

    K~_l = K^_l + sum_j P_lj K^_theta(x_j)                       (Eq. 1)
    minimise  sum_l (2l+1) C_l^input (K_l - K~_l)^2              (Eq. 2, C_l^input = 1: uncorrelated noise)
    A = [ delta_(l,l') for l' < l_cut | P_lj ],  W = diag(2l+1)  (Eq. 3-5), solved by SVD with singular values
    below `svd_cut` (relative to the largest) dropped

The real-space part is represented by its values at the n nodes x_j of the convolution library's table
(uniform in x = cos(theta) on [cos(theta_cut), 1]) and P_lj = 2 pi w_j P_l(x_j) with trapezoid weights w_j, i.e. the
Legendre transform b_l = 2 pi int K(x) P_l(x) dx of the piecewise-linear interpolant's samples (R3).
"""
import numpy as np


def legendre_matrix(lmax, x):
    """P[l, j] = P_l(x_j), l = 0 .. lmax, by the three-term recurrence (fp64)."""
    x = np.asarray(x, np.float64)
    P = np.empty((lmax + 1, x.size))
    P[0] = 1.0
    if lmax >= 1:
        P[1] = x
    for l in range(1, lmax):
        P[l + 1] = ((2 * l + 1) * x * P[l] - l * P[l - 1]) / (l + 1)
    return P


def gaussian_beam_ell(fwhm, lmax):
    """b_l of a unit-peak Gaussian beam exp(-theta^2 / 2 sigma^2) in the small-angle limit:
    2 pi sigma^2 exp(-l(l+1) sigma^2 / 2)."""
    sigma = fwhm / 2.3548
    l = np.arange(lmax + 1)
    return 2.0 * np.pi * sigma ** 2 * np.exp(-0.5 * l * (l + 1) * sigma ** 2)


def split_fit(K_ell, ell_cut, theta_cut, n_nodes, svd_cut=1e-6):
    """-> dict(K_hat_ell[ell_cut], K_hat_theta[n_nodes] at x_j = c + j (1-c)/(n-1), K_tilde_ell, sigma2_frac).

    sigma2_frac is Eq. 6 with alpha = 1: sum (2l+1)(K_l - K~_l)^2 / sum (2l+1) K_l^2."""
    K_ell = np.asarray(K_ell, np.float64)
    lmax = K_ell.size - 1
    if not (0 < ell_cut <= lmax + 1) or n_nodes < 2:
        raise ValueError("bad ell_cut / n_nodes")
    c = np.cos(theta_cut)
    x = c + np.arange(n_nodes) * (1.0 - c) / (n_nodes - 1)
    w = np.full(n_nodes, (1.0 - c) / (n_nodes - 1))
    w[0] *= 0.5
    w[-1] *= 0.5
    P = 2.0 * np.pi * legendre_matrix(lmax, x) * w[None, :]              # (lmax+1, n_nodes)
    A = np.zeros((lmax + 1, ell_cut + n_nodes))
    A[np.arange(ell_cut), np.arange(ell_cut)] = 1.0
    A[:, ell_cut:] = P
    sw = np.sqrt(2.0 * np.arange(lmax + 1) + 1.0)                        # sqrt(W): weighted least squares
    U, s, Vt = np.linalg.svd(A * sw[:, None], full_matrices=False)
    keep = s > svd_cut * s[0]
    xsol = Vt[keep].T @ ((U[:, keep].T @ (K_ell * sw)) / s[keep])
    K_tilde = A @ xsol
    num = np.sum((2.0 * np.arange(lmax + 1) + 1.0) * (K_ell - K_tilde) ** 2)
    den = np.sum((2.0 * np.arange(lmax + 1) + 1.0) * K_ell ** 2)
    return dict(x=x, K_hat_ell=xsol[:ell_cut], K_hat_theta=xsol[ell_cut:], K_tilde_ell=K_tilde,
                sigma2_frac=num / den, n_kept=int(keep.sum()))
