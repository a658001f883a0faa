"""The steps that close the chi^2 algorithm around the map (eq. 11) through the C ABI: each stage bit for
bit against oracle/chi2.py on oracle-made inputs, and the whole chain -- lt_gradient_points_sie ->
lt_source_barycentres -> lt_gradient_grid_sie -> lt_find_images -> lt_chi2, one stream, no host round trip -- against
the oracle's chain and the closed form of the singular isothermal sphere."""
import numpy as np
import pytest

from paper_1902_03252_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_1902_03252_b200 import lt
    from oracle import chi2 as C
    from oracle import find_images as FI
    from oracle import lt_oracle_sie as S
    lt.lib()
    return torch, lt, C, FI, S


def _catalogue(rng, n_systems, with_empty=True):
    counts = rng.integers(2, 6, n_systems)
    if with_empty:
        counts[rng.integers(0, n_systems, 3)] = 0
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    return offsets, int(offsets[-1])


def _hits_dev(torch, lt, source, x, y):
    rec = np.zeros(len(source), dtype=np.dtype(lt.HIT_DTYPE))
    rec["source"], rec["x"], rec["y"] = source, x, y
    rec["cell"] = np.arange(len(source))
    hits = torch.from_numpy(rec.view(np.uint8).reshape(-1, 32).copy()).cuda() if len(source) else \
        torch.zeros((1, 32), dtype=torch.uint8, device="cuda")
    return hits, torch.tensor([len(source)], dtype=torch.int32, device="cuda")


def test_stages_bit_for_bit(env):
    torch, lt, C, FI, S = env
    rng = np.random.default_rng(11)
    for n_sys in (1, 40, 300):
        offsets, n_img = _catalogue(rng, n_sys, with_empty=n_sys > 3)
        theta = rng.uniform(-60, 60, (n_img, 2))
        alpha = rng.normal(0, 9, (n_img, 2))
        ref = C.source_barycentres(theta, alpha, offsets, 0.731)
        got = lt.lt_source_barycentres(torch.from_numpy(theta).cuda(), torch.from_numpy(alpha).cuda(),
                                       torch.from_numpy(offsets).cuda(), 0.731).cpu().numpy()
        assert np.array_equal(got, ref, equal_nan=True)
        # predicted images: 0-4 per system, some systems with none, in shuffled order (the order of d_hits is not fixed)
        n_pred = rng.integers(0, 5, n_sys)
        src = rng.permutation(np.repeat(np.arange(n_sys), n_pred))
        hx, hy = rng.uniform(-60, 60, len(src)), rng.uniform(-60, 60, len(src))
        sigma = rng.uniform(0.05, 0.5, n_img)
        total, matched, unmatched, terms = C.chi2(theta, sigma, offsets, src, hx, hy)
        hits, n_hits = _hits_dev(torch, lt, src, hx, hy)
        res, t = lt.lt_chi2(torch.from_numpy(theta).cuda(), torch.from_numpy(sigma).cuda(), torch.from_numpy(offsets).cuda(),
                            hits, n_hits)
        assert lt.chi2_to_python(res) == (total, matched, unmatched)
        assert np.array_equal(t.cpu().numpy(), terms, equal_nan=True)
    # nothing observed: chi^2 = 0; n_hits beyond the capacity of d_hits: only the stored records count
    res, _ = lt.lt_chi2(torch.zeros((0, 2), dtype=torch.float64, device="cuda"), torch.zeros(0, dtype=torch.float64, device="cuda"),
                        torch.zeros(1, dtype=torch.int32, device="cuda"), hits, n_hits)
    assert lt.chi2_to_python(res) == (0.0, 0, 0)
    hits2, _ = _hits_dev(torch, lt, np.array([0, 0]), np.array([1.0, 50.0]), np.array([0.0, 0.0]))
    over = torch.tensor([7], dtype=torch.int32, device="cuda")
    res, _ = lt.lt_chi2(torch.tensor([[0.0, 0.0]], dtype=torch.float64, device="cuda"),
                        torch.tensor([0.5], dtype=torch.float64, device="cuda"),
                        torch.tensor([0, 1], dtype=torch.int32, device="cuda"), hits2, over)
    assert lt.chi2_to_python(res) == (4.0, 1, 0)


def test_chain_on_one_stream_against_the_oracle_chain_and_the_sis_closed_form(env):
    torch, lt, C, FI, S = env
    b0, delta, sigma = 2.0, 0.04, 0.1
    rng = np.random.default_rng(12)
    # several sources inside the Einstein radius of one SIS, each with its two images (closed form), one system per source
    beta = rng.uniform(-0.8, 0.8, (6, 2))
    u = beta / np.hypot(beta[:, 0], beta[:, 1])[:, None]
    obs = np.stack([beta + b0 * u, beta - b0 * u], axis=1).reshape(-1, 2)
    offsets = (2 * np.arange(7)).astype(np.int32)
    sig = np.full(12, sigma)
    model = np.array([[0.0, 0.0, 0.0, 0.0, b0 + delta]])
    n, dx = 321, 0.02
    x_min = -(n - 1) / 2 * dx - dx / 2
    # the oracle's chain
    a_ref = S.gradient_points(model, obs[:, 0], obs[:, 1])
    bary_ref = C.source_barycentres(obs, a_ref, offsets, 1.0)
    g_ref = S.gradient_grid(model, x_min, x_min, dx, n, n)
    h_ref = FI.find_images(g_ref, x_min, x_min, dx, 1.0, bary_ref)
    total_ref, m_ref, u_ref, terms_ref = C.chi2(obs, sig, offsets, h_ref["source"], h_ref["x"], h_ref["y"])
    # the library's chain: five calls on one side stream, one synchronisation at the end
    st = torch.cuda.Stream()
    L = torch.from_numpy(model).cuda()
    d_obs, d_sig, d_off = torch.from_numpy(obs).cuda(), torch.from_numpy(sig).cuda(), torch.from_numpy(offsets).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        alpha = lt.lt_gradient_points_sie(L, d_obs, stream=st)
        bary = lt.lt_source_barycentres(d_obs, alpha, d_off, 1.0, stream=st)
        g = lt.lt_gradient_grid_sie(L, x_min, x_min, dx, n, n, lt.LT_FP64, stream=st)
        hits, n_hits = lt.lt_find_images(g, x_min, x_min, dx, 1.0, bary, stream=st)
        res, terms = lt.lt_chi2(d_obs, d_sig, d_off, hits, n_hits, stream=st)
    st.synchronize()
    total, matched, unmatched = lt.chi2_to_python(res)
    assert (matched, unmatched) == (m_ref, u_ref) == (12, 0)
    assert np.abs(bary.cpu().numpy() - beta).max() < 1e-14
    assert abs(total / total_ref - 1) < 1e-9 and np.abs(terms.cpu().numpy() / terms_ref - 1).max() < 1e-9
    assert abs(total / (12 * delta ** 2 / sigma ** 2) - 1) < 2e-3          # closed form: delta^2 / sigma^2 per image
    print("chi2 chain: gpu %.12g oracle %.12g closed form %.12g" % (total, total_ref, 12 * delta ** 2 / sigma ** 2))
    # the same on the mixed-precision map (the paper's proposal): the predicted images barely move
    gm = lt.lt_gradient_grid_sie(L, x_min, x_min, dx, n, n, lt.LT_MIXED)
    hits_m, n_hits_m = lt.lt_find_images(gm, x_min, x_min, dx, 1.0, bary)
    res_m, terms_m = lt.lt_chi2(d_obs, d_sig, d_off, hits_m, n_hits_m)
    total_m, matched_m, unmatched_m = lt.chi2_to_python(res_m)
    moved = sigma * np.abs(np.sqrt(terms_m.cpu().numpy()) - np.sqrt(terms.cpu().numpy())).max()
    print("chi2 chain on the mixed map: %.12g, image distances change by at most %.2e arcsec" % (total_m, moved))
    assert (matched_m, unmatched_m) == (12, 0) and abs(total_m / total - 1) < 1e-3 and moved < 1e-3 * dx
