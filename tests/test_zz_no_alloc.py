"""wolff_energy_magnetisation_noalloc against wolff_observables.

Why the entry point exists: a program that already holds its lattice on the GPU may be unable to let a library
allocate there -- it gave the whole card to its own arena when it started, or it must stay inside a memory budget fixed
at start-up, or it has a latency-critical loop on other streams that a cudaMalloc / cudaFree would stall.  Every other
call of this library needs a handle, and making a handle allocates.  The no-allocation call takes the caller's lattice
and two caller-owned result words and keeps its scratch (per-CTA partial sums, a ticket) in a fixed array inside the
library image, which is why it refuses lattices above NOALLOC_MAX_SITES.

What is checked: on the same lattice bytes the new call returns exactly the E and M the existing path returns
(tolerance: none -- both are integer sums, like every other GPU test here), on TWO calls in a row that are queued on
one stream without a synchronisation between them and work on different lattices: the second call finds the scratch
array as the first one left it, so a ticket that is not cleared, or a stale slot that is read, shows up as a wrong sum.
The lattices cover both kernels (L a multiple of 16 or not), one CTA and many, a ragged last CTA, 2D and 3D, and the
largest size allowed.

This file is named to be collected last: it does not depend on the other tests, and a failure here must not hide theirs
under `pytest -x`.
"""
import numpy as np
import pytest

from paper_1110_0899_b200 import binding
from paper_1110_0899_b200 import workloads as wl


def test_sizes_beyond_the_scratch_array_are_refused_before_any_cuda_call():
    """The limit is checked first, so a caller learns about it even on a machine without a GPU."""
    lib = binding.load()
    for dim, L in [(2, 16385), (3, 646), (2, 1 << 20), (3, 4096)]:
        assert L ** dim > binding.NOALLOC_MAX_SITES
        assert lib.wolff_energy_magnetisation_noalloc(16, dim, L, 16, 32, None) == binding.WOLFF_EINVAL
        assert "WOLFF_NOALLOC_MAX_SITES" in binding.last_error()
    for dim, L in [(1, 8), (4, 8), (2, 1), (2, 0), (3, -5)]:
        assert lib.wolff_energy_magnetisation_noalloc(16, dim, L, 16, 32, None) == binding.WOLFF_EINVAL
    assert lib.wolff_energy_magnetisation_noalloc(None, 2, 8, 16, 32, None) == binding.WOLFF_EINVAL
    assert lib.wolff_energy_magnetisation_noalloc(8, 2, 16, 16, 32, None) == binding.WOLFF_EINVAL      # misaligned for L % 16 == 0
    assert 16385 ** 2 > binding.NOALLOC_MAX_SITES >= 16384 ** 2 and 646 ** 3 > binding.NOALLOC_MAX_SITES >= 645 ** 3


CASES = [  # dim, L, T, updates between the two snapshots
    (2, 2, 2.0, 3), (2, 3, 2.0, 3), (3, 2, 4.0, 3), (3, 3, 4.0, 3),           # every bond wraps
    (2, 16, wl.TC_2D, 5), (2, 64, wl.TC_2D, 20),                               # vector kernel, one CTA, partly filled
    (2, 100, 2.0, 20), (3, 30, 4.0, 20),                                       # scalar kernel, ragged last CTA
    (2, 1024, wl.TC_2D, 30), (3, 64, wl.TC_3D, 30),                            # vector kernel, 64 and 16 CTAs
    (2, 1040, 2.2, 10), (3, 48, 4.4, 10),                                      # vector kernel, ragged last CTA
    (2, 4096, wl.TC_2D, 4), (3, 256, wl.TC_3D, 4),                             # the BASELINE lattices: 1024 CTAs
    (3, 250, 4.3, 3),                                                          # scalar kernel, 954 CTAs
]


def _snapshot(chain, torch):
    """(device copy of the chain's lattice, E and M of it by the existing path)."""
    spins = torch.empty(chain.N, dtype=torch.int8, device="cuda")
    chain.get_spins_into(spins)
    return spins, chain.observables()


@pytest.mark.gpu
@pytest.mark.parametrize("dim,L,T,n", CASES)
def test_two_calls_in_a_row_match_the_existing_path(dim, L, T, n):
    import torch
    with binding.Wolff(dim, L, 1.0, T, seed=1234 + L) as chain:
        first, want_first = _snapshot(chain, torch)
        chain.run(n)
        second, want_second = _snapshot(chain, torch)
    out = torch.full((4,), -(1 << 62), dtype=torch.int64, device="cuda")
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    # two calls back to back on one stream, no synchronisation in between
    binding.energy_magnetisation_noalloc(first, dim, L, out[0:1], out[1:2], stream)
    binding.energy_magnetisation_noalloc(second, dim, L, out[2:3], out[3:4], stream)
    stream.synchronize()
    got = out.cpu().tolist()
    assert (got[0], got[1]) == want_first, "first call"
    assert (got[2], got[3]) == want_second, "second call (scratch left behind by the first)"
    # and against the definition, with numpy, for the lattices where that is cheap
    if L ** dim <= 1 << 21:
        s = second.cpu().numpy().astype(np.int64).reshape((L,) * dim)
        E = -sum(int((s * np.roll(s, -1, axis=a)).sum()) for a in range(dim))
        assert (E, int(s.sum())) == (got[2], got[3])


@pytest.mark.gpu
def test_largest_lattice_null_outputs_pinned_host_output_and_wrong_memory():
    import torch
    L = 16384                                            # N = 2^28 = NOALLOC_MAX_SITES: all 16,384 slots in use
    with binding.Wolff(2, L, 1.0, 2.4, seed=99) as chain:
        spins, want = _snapshot(chain, torch)
    assert spins.numel() == binding.NOALLOC_MAX_SITES
    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    pinned = torch.zeros(2, dtype=torch.int64).pin_memory()
    binding.energy_magnetisation_noalloc(spins, 2, L, out[0:1], None)          # E only
    binding.energy_magnetisation_noalloc(spins, 2, L, None, out[1:2])          # M only
    binding.energy_magnetisation_noalloc(spins, 2, L, pinned[0:1], pinned[1:2])
    binding.energy_magnetisation_noalloc(spins, 2, L, None, None)              # nothing asked for: a no-op
    torch.cuda.synchronize()
    assert tuple(out.cpu().tolist()) == want
    assert tuple(pinned.tolist()) == want
    # a lattice in pageable host memory is refused (there is no staging copy: that would need an allocation)
    host = np.ones(64 * 64, dtype=np.int8)
    with pytest.raises(binding.WolffError) as err:
        binding.energy_magnetisation_noalloc(host, 2, 64, out[0:1], out[1:2])
    assert err.value.code == binding.WOLFF_EINVAL
    # the refused call left the library usable
    small = torch.ones(64 * 64, dtype=torch.int8, device="cuda")
    binding.energy_magnetisation_noalloc(small, 2, 64, out[0:1], out[1:2])
    torch.cuda.synchronize()
    assert tuple(out.cpu().tolist()) == (-2 * 64 * 64, 64 * 64)
