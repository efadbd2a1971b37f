"""smcx_pair_counts_static (include/smcx.h): the pair counts of Eq. 8 (reading S7) through the entry
point that allocates no device memory -- its accumulator is a file-scope device array of the library -- against the
existing path (smcx_sro, accumulator in the handle's workspace) and the oracle, on two calls in a row.  Integer counts:
the bar is bit-exact.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import paper_2509_20949_b200 as smcx
from smcx_inputs import make_accept_table, make_epi

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("lattice,dims,n_sp,n_sh", [
    (smcx.BCC, (16, 24, 8), 4, 2),     # the graded configuration's lattice in small (2-bit storage on the existing path)
    (smcx.FCC, (16, 8, 16), 5, 3),     # config 3's lattice in small
    (smcx.BCC, (8, 8, 16), 16, 4),     # 4 x 256 = 1,024 entries: exactly the size of the static scratch
])
def test_static_pair_counts_match_the_existing_path_on_two_calls_in_a_row(lattice, dims, n_sp, n_sh):
    import torch
    import oracle
    seed = 321
    epi, table = make_epi(n_sh, n_sp, 300, seed), make_accept_table(860)
    g = smcx.Lattice(lattice, dims, n_sp, n_sh, epi, table, seed, link_cell=4, kT_units=860)
    o = oracle.Oracle(lattice, dims, n_sp, n_sh, epi, 4, table, seed)
    out = torch.full((n_sh, n_sp, n_sp), -7, dtype=torch.int64, device="cuda")     # stale contents must be overwritten
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    for call in range(2):
        g.sweep(2)                                        # a different state for the second call
        o.sweep(2)
        _, want = g.sro()                                 # existing path: accumulator in the handle's workspace
        species = g.species_device()                      # the caller's input: uint8 device tensor
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        with torch.cuda.stream(stream):
            got = smcx.pair_counts_static(lattice, dims, n_sp, n_sh, species, out, stream=stream)
        stream.synchronize()
        if call == 1:                                     # the first call may load the module lazily
            assert torch.cuda.mem_get_info()[0] >= free_before, "the no-alloc entry point took device memory"
        got = got.cpu().numpy()
        assert (got == want).all(), f"call {call}: static-scratch pair counts differ from smcx_sro"
        assert (got == o.sro()[1]).all(), f"call {call}: static-scratch pair counts differ from the oracle"
        assert got.sum() > 0 and (got == got.transpose(0, 2, 1)).all()
    g.close()


def test_static_pair_counts_default_stream_and_smaller_problem_after_a_larger_one():
    """The array keeps the last call's contents: a small problem right after a large one must not see them."""
    import torch
    rng = np.random.default_rng(5)
    big = torch.from_numpy(rng.integers(0, 16, 2 * 8 * 8 * 8, dtype=np.uint8)).cuda()
    out_big = torch.empty((4, 16, 16), dtype=torch.int64, device="cuda")
    smcx.pair_counts_static(smcx.BCC, (8, 8, 8), 16, 4, big, out_big)
    epi, table = make_epi(1, 2, 300, 9), make_accept_table(600)
    g = smcx.Lattice(smcx.BCC, (8, 8, 8), 2, 1, epi, table, 9, link_cell=4, kT_units=600)
    _, want = g.sro()
    out = torch.empty((1, 2, 2), dtype=torch.int64, device="cuda")
    smcx.pair_counts_static(smcx.BCC, (8, 8, 8), 2, 1, g.species_device(), out)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == want).all()
    assert int(out_big.sum().item()) == 2 * 8 * 8 * 8 * (8 + 6 + 12 + 24)       # every site, every neighbour of 4 BCC shells
    g.close()


def test_static_pair_counts_reject_what_does_not_fit():
    import torch
    sp = torch.zeros(2 * 8 * 8 * 8, dtype=torch.uint8, device="cuda")
    out = torch.zeros((5, 16, 16), dtype=torch.int64, device="cuda")
    assert 5 * 16 * 16 > smcx.STATIC_PAIR_COUNTS_MAX
    with pytest.raises(smcx.SmcxError) as e:
        smcx.pair_counts_static(smcx.BCC, (8, 8, 8), 16, 5, sp, out)
    assert e.value.code == -15 and "1024" in str(e.value)
    for bad in (dict(lattice=2), dict(dims=(8, 1, 8)), dict(n_species=1), dict(n_species=17), dict(n_shells=0), dict(n_shells=6)):
        kw = dict(lattice=smcx.BCC, dims=(8, 8, 8), n_species=4, n_shells=2)
        kw.update(bad)
        with pytest.raises(smcx.SmcxError):
            smcx.pair_counts_static(kw["lattice"], kw["dims"], kw["n_species"], kw["n_shells"], sp, out)
    torch.cuda.synchronize()
    assert int(out.abs().sum().item()) == 0                     # out-parameters are written only on success
