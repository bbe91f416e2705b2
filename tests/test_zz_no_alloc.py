"""te_nuclear_attraction_noalloc (the allocation-free entry point: static device scratch, nbf <= 512) against the existing
te_nuclear_attraction path, on two calls in a row.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_noalloc_nuclear_attraction_matches_existing_path_twice():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2406_14920_b200 as te
    from synth import make_config
    for n in (2, 1):                                   # nbf 504 (close to the 512 limit, all 10 pair classes), then nbf 80
        prob = make_config(n)
        b = te.Basis.from_problem(prob)
        pr = b.shellpair_build(prob.tau_pair)
        rng = np.random.default_rng(1426 + n)
        V = torch.full((b.nbf, b.nbf), 7.0, dtype=torch.float64, device="cuda")      # overwritten, not accumulated
        for call in range(2):                          # second call: other charges; the scratch must not keep the first result
            m = min(5 + 3 * call, prob.natoms - call)
            xyz = np.vstack([prob.xyz[:m], rng.uniform(-3.0, 9.0, (2, 3))])
            q = np.concatenate([-rng.uniform(1.0, 8.0, m), [0.4, -2.0]])
            ref = pr.nuclear_attraction(xyz, q).cpu().numpy()                        # existing path (allocates)
            xyzq = torch.tensor(np.hstack([xyz, q[:, None]]), device="cuda")
            torch.cuda.synchronize()
            before = torch.cuda.memory_allocated()
            pr.nuclear_attraction_noalloc(xyzq, V)
            torch.cuda.synchronize()
            assert torch.cuda.memory_allocated() == before
            got = V.cpu().numpy()
            scale = max(1.0, float(np.max(np.abs(ref))))
            assert np.max(np.abs(got - ref)) <= 1e-11 * scale, (n, call, float(np.max(np.abs(got - ref))))
            assert np.max(np.abs(got - got.T)) == 0.0
        pr.nuclear_attraction_noalloc(torch.zeros((0, 4), dtype=torch.float64, device="cuda"), V)   # no charges: zero matrix
        torch.cuda.synchronize()
        assert float(V.abs().max()) == 0.0
    # beyond the static scratch: a clear error, nothing launched
    prob = make_config(3)                              # nbf 768 > 512
    b = te.Basis.from_problem(prob)
    pr = b.shellpair_build(prob.tau_pair)
    V = torch.zeros((b.nbf, b.nbf), dtype=torch.float64, device="cuda")
    with pytest.raises(te.TEError, match="TE_NOALLOC_MAX_NBF"):
        pr.nuclear_attraction_noalloc(torch.zeros((1, 4), dtype=torch.float64, device="cuda"), V)
