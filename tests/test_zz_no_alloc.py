"""phoebe_elph_set_k_noalloc: the allocation-free variant of set_k (a1 + a2, Eq. 71) whose scratch tensor
lives in a fixed file-scope device array inside the library (include/phoebe_elph.h, csrc/noalloc.cu).

Checked against the existing context-based path (phoebe_elph_set_k + phoebe_elph_copy_g1) on the same inputs, on TWO
calls in a row that share the scratch array (different k, different shapes: the second call is smaller, so stale contents
of the first would show), within the tolerance the other GPU tests use for g1' (1e-12 relative; the two paths sum the Re
list in a different order), and against the CPU oracle.  The file name sorts last on purpose: the run uses
`pytest -x`, and a failure here must not hide the other tests.  Passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_G1 = 1e-12


def _relerr(got, ref):
    return float(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))


@pytest.fixture(scope="module")
def env():
    import torch
    import oracle
    from paper_2111_14999_b200 import binding, build, harness, workloads as wl
    build.build()
    binding.load_library()
    assert torch.cuda.is_available()
    binding.noalloc_setup()                      # once per device, outside anything that forbids allocation
    # one tiny warm-up call: the CUDA runtime loads a kernel's code on its first launch (lazy module loading)
    z = lambda *shape, dt=torch.complex128: torch.zeros(shape, dtype=dt, device="cuda")
    binding.set_k_noalloc(z(1, 1, 1, 1, 1), z(1, 3, dt=torch.float64), None, (0.0, 0.0, 0.0), z(1, 1), z(1, 1, 1, 1))
    torch.cuda.synchronize()
    return dict(torch=torch, oracle=oracle, binding=binding, harness=harness, wl=wl)


def _existing_path(env, w, gW_d, k, Uk, deg_e=None):
    harness = env["harness"]
    ctx = harness.make_context(w, gW_d, nq_max=64, deg_e=deg_e)
    ctx.set_k(k, harness.to_device([Uk])[0])
    g1 = ctx.copy_g1().cpu().numpy()
    ctx.close()
    return g1


def test_no_alloc_matches_existing_path_on_two_calls_in_a_row(env):
    torch, oracle, binding, harness, wl = (env[k] for k in ("torch", "oracle", "binding", "harness", "wl"))
    # first call: 45 x 5 x 5 x 6 = 6750 complex of scratch; second call: smaller in every dimension, with degeneracies
    w1 = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(5, 4, 3), grid_p=(5, 3, 3), nk=2, nq=8, cfg_id=210)
    w2 = wl.custom(nw=3, nb1=3, nb2=3, nm=3, grid_e=(7, 11, 9), grid_p=(2, 2, 3), nk=2, nq=8, cfg_id=211)   # 693 Re: two phase chunks
    cases = []
    for w, ik, with_deg in ((w1, 0, False), (w2, 1, True)):
        gW = wl.gW_full(w)
        deg_e = np.random.default_rng(5).integers(1, 4, w.nRe).astype(np.float64) if with_deg else None
        cases.append(dict(w=w, gW=gW, gW_d=torch.from_numpy(gW).cuda(), Re=wl.Re_vectors(w), k=wl.k_points(w)[ik],
                          Uk=wl.U_k(w, ik), deg_e=deg_e))
    # inputs and outputs are the caller's: allocated BEFORE the calls
    for c in cases:
        c["Re_d"], c["Uk_d"] = harness.to_device([c["Re"], c["Uk"]])
        c["deg_d"] = harness.to_device([c["deg_e"]])[0] if c["deg_e"] is not None else None
        c["out_d"] = torch.full((c["w"].nRp, c["Uk"].shape[1], c["w"].nw, c["w"].nm), float("nan"), dtype=torch.complex128,
                                device="cuda")
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    stats0 = torch.cuda.memory_stats().get("allocation.all.allocated", 0)
    for c in cases:                               # two calls in a row on the same stream: they share the scratch array
        binding.set_k_noalloc(c["gW_d"], c["Re_d"], c["deg_d"], c["k"], c["Uk_d"], c["out_d"])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_stats().get("allocation.all.allocated", 0) == stats0   # nothing was allocated
    for c in cases:
        got = c["out_d"].cpu().numpy()
        assert np.all(np.isfinite(got.view(np.float64)))
        ref_gpu = _existing_path(env, c["w"], c["gW_d"], c["k"], c["Uk"], c["deg_e"])
        ref_cpu = oracle.setk(c["gW"], c["Re"], c["deg_e"], c["k"], c["Uk"])
        assert got.shape == ref_gpu.shape
        assert _relerr(got, ref_gpu) <= TOL_G1
        assert _relerr(got, ref_cpu) <= TOL_G1
    # and once more the first problem after the second: the result does not depend on what the array held
    c = cases[0]
    first = c["out_d"].cpu().numpy().copy()
    c["out_d"].fill_(float("nan"))
    binding.set_k_noalloc(c["gW_d"], c["Re_d"], c["deg_d"], c["k"], c["Uk_d"], c["out_d"])
    assert np.array_equal(c["out_d"].cpu().numpy(), first)


def test_no_alloc_rejects_sizes_beyond_the_fixed_scratch(env):
    torch, binding = env["torch"], env["binding"]
    nRp, nRe, nw, nm = 1, 1, 16, 1025                     # 16 x 16 x 1025 x 16 B = 4.2 MB > 4 MiB
    assert nRp * nw * nw * nm * 16 > binding.NOALLOC_MAX_BYTES
    gW = torch.zeros((nRp, nRe, nw, nw, nm), dtype=torch.complex128, device="cuda")
    Re = torch.zeros((nRe, 3), dtype=torch.float64, device="cuda")
    Uk = torch.zeros((nw, 2), dtype=torch.complex128, device="cuda")
    out = torch.zeros((nRp, 2, nw, nm), dtype=torch.complex128, device="cuda")
    with pytest.raises(binding.PhoebeElphError) as ei:
        binding.set_k_noalloc(gW, Re, None, (0.1, 0.2, 0.3), Uk, out)
    assert ei.value.code == -2 and "exceed the fixed scratch" in str(ei.value) and "4194304" in str(ei.value)
    # exactly at the limit is accepted: 16 x 16 x 1024 complex = 4 MiB
    nm = 1024
    gW = torch.ones((nRp, nRe, nw, nw, nm), dtype=torch.complex128, device="cuda")
    Uk = torch.zeros((nw, 2), dtype=torch.complex128, device="cuda"); Uk[0, 0] = 1.0; Uk[1, 1] = 2.0
    out = torch.zeros((nRp, 2, nw, nm), dtype=torch.complex128, device="cuda")
    binding.set_k_noalloc(gW, Re, None, (0.1, 0.2, 0.3), Uk, out)        # R = 0: phase 1, T = g_W
    got = out.cpu().numpy()
    assert np.allclose(got[0, 0], 1.0) and np.allclose(got[0, 1], 2.0)
    with pytest.raises(binding.PhoebeElphError) as ei:                   # nb1 > nw
        binding.set_k_noalloc(gW, Re, None, (0.0, 0.0, 0.0), torch.zeros((nw, nw + 1), dtype=torch.complex128, device="cuda"),
                              torch.zeros((nRp, nw + 1, nw, nm), dtype=torch.complex128, device="cuda"))
    assert ei.value.code == -2
