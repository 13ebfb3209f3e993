"""mk_image_static (include/mk.h): the imaging call whose scratch is a static device array, for callers that cannot call
cudaMalloc.  Checked against the existing path (mk_image, which takes its scratch from the context) on the same fields,
on calls in a row that share the array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import oracle
from paper_2106_04649_b200 import configs
from _util import calibrated, problem, rel_l2

pytestmark = pytest.mark.gpu

TOL_FINAL = 1e-4   # the tolerance of the final fields in tests/test_parity_gpu.py


def _run_and_image(mk, B, cfg, dev):
    """One run on `mk`; returns (Gminus, f1plus, image by the existing path) as device tensors."""
    import torch
    R, Gd, td = problem(cfg)
    mk.load_R(torch.from_numpy(R).to(dev))
    outs = {nm: torch.empty((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in ("Gminus", "f1plus")}
    mk.run(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev), cfg.niter, outs)
    img = torch.empty(cfg.nfoc, dtype=torch.float32, device=dev)
    mk.image(outs["Gminus"], img)
    return outs["Gminus"], outs["f1plus"], img


def test_image_static_equals_mk_image_on_calls_in_a_row():
    import torch
    from paper_2106_04649_b200 import binding as B
    dev = torch.device("cuda:0")
    big = calibrated(configs.scaled(2, n=48, nt=256, nfoc=48, focal="line:300", niter=4))
    small = calibrated(configs.scaled(2, n=40, nt=128, nfoc=5, focal="fan:300", niter=3))
    with B.Marchenko(big.n, big.n, big.nt, big.dt, big.dx, big.fmin, big.fmax) as mk_a, \
            B.Marchenko(small.n, small.n, small.nt, small.dt, small.dx, small.fmin, small.fmax) as mk_b:
        for mk, cfg in ((mk_a, big), (mk_b, small)):
            mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
        ga, pa, img_a = _run_and_image(mk_a, B, big, dev)
        gb, pb, img_b = _run_and_image(mk_b, B, small, dev)
        assert float(img_a.abs().max()) > 0 and float(img_b.abs().max()) > 0
        torch.cuda.synchronize()
        # big, then small (the array still holds the big call's sums beyond the small call's), then big again
        got = []
        for k, (mk, g, p, nfoc) in enumerate(((mk_a, ga, pa, big.nfoc), (mk_b, gb, pb, small.nfoc), (mk_a, ga, pa, big.nfoc))):
            out = torch.full((nfoc,), float("nan"), dtype=torch.float32, device=dev)
            bytes_before = mk.get_info(B.MK_INFO_DEVICE_BYTES)
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info(dev)[0]
            mk.image_static(g, p, out)
            torch.cuda.synchronize()
            if k > 0:   # the first call on the device may load the module lazily; no later call may take device memory
                assert torch.cuda.mem_get_info(dev)[0] >= free_before
            assert mk.get_info(B.MK_INFO_DEVICE_BYTES) == bytes_before
            got.append(out.cpu().numpy())
        for out, ref in zip(got, (img_a, img_b, img_a)):
            ref = ref.cpu().numpy()
            e = rel_l2(out, ref)
            print(f"\n[image_static nfoc={len(ref)}] rel L2 against mk_image {e:.2e}")
            assert e <= TOL_FINAL
            np.testing.assert_array_equal(out, ref)   # same kernels, same grid, fixed order of summation


def test_image_static_needs_no_run_and_matches_the_oracle_at_the_limit():
    """nfoc = MK_IMAGE_STATIC_MAX_PARTIALS with two receivers fills the array exactly (one chunk per focal point)."""
    import torch
    from paper_2106_04649_b200 import binding as B
    dev = torch.device("cuda:0")
    n, nt, dt, dx = 2, 64, 0.004, 10.0
    nfoc = B.MK_IMAGE_STATIC_MAX_PARTIALS
    rng = np.random.default_rng(20210649)
    g = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    p = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    ref = oracle.image(g, p, dt, dx)
    with B.Marchenko(n, n, nt, dt, dx, 5.0, 60.0) as mk:
        out = torch.empty(nfoc, dtype=torch.float32, device=dev)
        for _ in range(2):
            out.fill_(float("nan"))
            mk.image_static(torch.from_numpy(g).to(dev), torch.from_numpy(p).to(dev), out)
            e = rel_l2(out.cpu().numpy(), ref)
            assert e <= 2e-6, e   # fp32 products, fp32 sums of 64 terms, double across receivers


def test_image_static_rejects_sizes_beyond_the_static_array():
    import torch
    from paper_2106_04649_b200 import binding as B
    dev = torch.device("cuda:0")
    n, nt = 2, 64
    nfoc = B.MK_IMAGE_STATIC_MAX_PARTIALS + 1
    with B.Marchenko(n, n, nt, 0.004, 10.0, 5.0, 60.0) as mk:
        g = torch.ones((nfoc, n, nt), dtype=torch.float32, device=dev)
        out = torch.full((nfoc,), 7.0, dtype=torch.float32, device=dev)
        launches = mk.get_info(B.MK_INFO_KERNEL_LAUNCHES)
        with pytest.raises(B.MkError) as ei:
            mk.image_static(g, g, out)
        assert ei.value.code == B.MK_ERR_INVALID_ARG
        assert "MK_IMAGE_STATIC_MAX_PARTIALS" in str(ei.value) and str(nfoc) in str(ei.value)
        assert mk.get_info(B.MK_INFO_KERNEL_LAUNCHES) == launches      # nothing was launched
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())
        # the context is still usable, and a size within the limit goes through afterwards
        ok = torch.empty(3, dtype=torch.float32, device=dev)
        mk.image_static(g[:3].contiguous(), g[:3].contiguous(), ok)
        # G^- = f1plus = 1: sum_j 1 = nt per receiver, both receivers are end points of the trapezoid rule (weight dx / 2)
        np.testing.assert_allclose(ok.cpu().numpy(), 0.004 * (10.0 * 0.5) * 2 * nt, rtol=1e-6)
