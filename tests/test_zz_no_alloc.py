"""ca_counts_noalloc: the entry point that allocates nothing (fixed device scratch inside the library) against the existing
path (ca_counts / ca_fitness on a context).  Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

from paper_2303_08123_b200 import binding, workloads as w

pytestmark = pytest.mark.gpu


def _state_tensor(g, torch):
    """the batch's exported state arrays as one cuda tensor [batch][nz][ny][nx] (the caller-owned input of the new entry point)"""
    host = np.stack([g.get_state(b, fields=False)["state"] for b in range(g.batch)])
    return torch.from_numpy(host).cuda()


def test_counts_noalloc_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    p = w.stress_params(N_ref=1500)
    dims = (24, 20, 12)
    B = 5
    g = binding.CaBatch(B, *dims, p, max_frac=2)
    g.seed("ball", radius=3.5, rng_seed=2024, sim_id_base=3)
    g.set_protocols(np.full((B, 1), 4.0), np.full((B, 1), 0.02))
    counts = torch.full((B, binding.CA_NCOUNT), -7, dtype=torch.int32, device="cuda")
    fit = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    seen = []
    for steps in (40, 60):                                     # two calls in a row: the second must not see the first one's sums
        g.step(steps)
        ref_c, ref_f = g.counts(), g.fitness()
        st = _state_tensor(g, torch)
        binding.counts_noalloc(st, *dims, n_ref=1500, counts_out=counts, fitness_out=fit)
        torch.cuda.synchronize()
        assert np.array_equal(counts.cpu().numpy(), ref_c)     # integers: bit-exact, as in every parity test
        assert np.array_equal(fit.cpu().numpy(), ref_f)
        seen.append(ref_c[:, 0].copy())
    assert not np.array_equal(seen[0], seen[1]) and (seen[1] > 0).all()          # the two calls really saw different lattices
    # a smaller batch after a larger one, fitness only, default N_ref (interior sites), on a stream of the caller's
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        f2 = torch.zeros(2, dtype=torch.float32, device="cuda")
        binding.counts_noalloc(st[3:5].contiguous(), *dims, fitness_out=f2, stream=s)
    s.synchronize()
    interior = (dims[0] - 2) * (dims[1] - 2) * (dims[2] - 2)
    assert np.array_equal(f2.cpu().numpy(), (interior - ref_c[3:5, 12]).astype(np.float32))
    g.close()


def test_counts_noalloc_rejects_what_the_fixed_scratch_cannot_hold():
    import torch
    L = binding.load()
    st = torch.zeros(64, dtype=torch.uint8, device="cuda")
    out = torch.zeros(16, dtype=torch.float32, device="cuda")
    vp = lambda t: C.c_void_p(t.data_ptr())
    rc = L.ca_counts_noalloc(vp(st), binding.CA_NOALLOC_MAX_BATCH + 1, 4, 4, 4, 0, None, vp(out), None)
    assert rc == binding.CA_EINVAL and b"CA_NOALLOC_MAX_BATCH" in L.ca_last_error(None)
    assert L.ca_counts_noalloc(vp(st), 1, 4, 4, 4, 0, None, None, None) == binding.CA_EINVAL          # no output
    assert L.ca_counts_noalloc(None, 1, 4, 4, 4, 0, None, vp(out), None) == binding.CA_EINVAL
    assert L.ca_counts_noalloc(C.c_void_p(st.data_ptr() + 4), 1, 4, 4, 4, 0, None, vp(out), None) == binding.CA_EINVAL   # misaligned
    with pytest.raises(binding.CaError):
        binding.counts_noalloc(torch.zeros((binding.CA_NOALLOC_MAX_BATCH + 1, 3, 3, 3), dtype=torch.uint8, device="cuda"), 3, 3, 3, fitness_out=out)
