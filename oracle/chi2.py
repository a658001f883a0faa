"""TEST INFRASTRUCTURE, NOT THE PRODUCT: plain numpy / Python-loop oracle for the two small steps that close the paper's
chi^2 algorithm around the deflection map (section 2.2.2; eq. 11) -- SURVEY 8(f) NEXT-3:

  "we loop over each multiple image j in each multiple image system i.  For each multiple image, we use equation 13 to
   compute the source coordinates, beta_ij,1 and beta_ij,2.  Subsequently, we determine the barycenter of the sources of a
   given multiple image system i."
  "Once we have found the locations of all predicted multiple images for all multiple image systems, we compute the
   chi^2 according to equation 11":   chi^2 = sum_i sum_j (x_obs,ij - x_ij)^2 / sigma_ij^2

Step by step, fp64, in the order written:
  source_barycentres:  beta_ij = theta_ij - (D_LS/D_OS) * alpha_ij   (eq. 13; product and difference rounded
                       separately), barycentre_i = (sum over j in catalogue order of beta_ij) / n_i.  A system without
                       images has no barycentre: (nan, nan).
  chi2:                for every observed image ij, x_ij = the predicted image of system i nearest to it (reading R28:
                       the paper does not say how predicted and observed images are paired), term_ij =
                       ((dx*dx + dy*dy) / (sigma*sigma)); chi^2 = sum of the terms in catalogue order.  An observed
                       image whose system has no predicted image has no term (nan) and is counted as unmatched
                       (reading R28: the paper does not say what such a model costs; the caller decides).
The images of system i are rows offsets[i] .. offsets[i+1]-1 of the catalogue.
Imports nothing from paper_1902_03252_b200.  Only tests/ may import it.
"""
import numpy as np


def source_barycentres(theta, alpha, offsets, dls_dos):
    theta = np.asarray(theta, dtype=np.float64).reshape(-1, 2)
    alpha = np.asarray(alpha, dtype=np.float64).reshape(-1, 2)
    offsets = np.asarray(offsets, dtype=np.int64)
    r = np.float64(dls_dos)
    out = np.full((len(offsets) - 1, 2), np.nan)
    for i in range(len(offsets) - 1):
        n = int(offsets[i + 1] - offsets[i])
        if n == 0:
            continue
        s1, s2 = np.float64(0.0), np.float64(0.0)
        for j in range(int(offsets[i]), int(offsets[i + 1])):
            s1 = s1 + (theta[j, 0] - r * alpha[j, 0])        # eq. 13
            s2 = s2 + (theta[j, 1] - r * alpha[j, 1])
        out[i, 0], out[i, 1] = s1 / np.float64(n), s2 / np.float64(n)
    return out


def chi2(theta_obs, sigma, offsets, hit_source, hit_x, hit_y):
    """Returns (chi2, n_matched, n_unmatched, terms[n_images]); hit_* describe the predicted images (source = system)."""
    theta_obs = np.asarray(theta_obs, dtype=np.float64).reshape(-1, 2)
    sigma = np.asarray(sigma, dtype=np.float64)
    offsets = np.asarray(offsets, dtype=np.int64)
    hit_source = np.asarray(hit_source)
    hit_x, hit_y = np.asarray(hit_x, dtype=np.float64), np.asarray(hit_y, dtype=np.float64)
    terms = np.full(len(theta_obs), np.nan)
    total, matched, unmatched = np.float64(0.0), 0, 0
    for i in range(len(offsets) - 1):
        mine = hit_source == i
        for j in range(int(offsets[i]), int(offsets[i + 1])):
            if not mine.any():
                unmatched += 1
                continue
            dx, dy = theta_obs[j, 0] - hit_x[mine], theta_obs[j, 1] - hit_y[mine]
            d2 = (dx * dx + dy * dy).min()                   # nearest predicted image of the same system
            terms[j] = d2 / (sigma[j] * sigma[j])            # eq. 11
            total = total + terms[j]
            matched += 1
    return float(total), matched, unmatched, terms
