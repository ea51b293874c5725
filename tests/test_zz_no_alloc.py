"""ising_energy_static (include/ising.h): E and M of a canonical packed sample with no handle, no workspace and no allocation --
the scratch is a fixed device array inside the library.  Collected last on purpose (the suite runs with pytest -x).

The expected values come from the existing path (ising_load_state + ising_energy on a handle with a caller workspace) and from the
oracle; all outputs are integers, tolerance 0 (R15).  Two calls in a row on different inputs, then the first input again:
the shared array keeps the previous call's contents, and nothing of it may show.
"""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import PHILOX, Ising, binding, synth  # noqa: E402


def dev(a: np.ndarray):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def test_static_entry_point_argument_checks_without_a_gpu():
    lib = binding.lib()
    one = C.c_void_p(256)   # never dereferenced: the checks come first
    assert lib.ising_energy_static(64, None, one, one, one, None) == binding.EINVAL
    assert lib.ising_energy_static(64, one, one, None, one, None) == binding.EINVAL
    for L in (0, 16, 62, 96, 100):
        assert lib.ising_energy_static(L, one, one, one, one, None) == binding.EINVAL, L
    for L in (192, 256, 1024):
        assert lib.ising_energy_static(L, one, one, one, one, None) == binding.ELIMIT, L
    assert b"ISING_STATIC_MAX_L" in lib.ising_strerror(binding.ELIMIT)
    assert binding.STATIC_MAX_L == 128


@pytest.mark.gpu
@pytest.mark.parametrize("L", [64, 128])
def test_static_energy_equals_the_handle_path_on_two_calls_in_a_row(L):
    inputs = [(synth.make_spins(L, 1, 41 + k), synth.make_couplings(L, 1, 51 + k)) for k in range(2)]
    want = []
    for spins, J in inputs:
        g = Ising(L, 1, synth.DYN_SEED, PHILOX)
        g.ising_load_state(dev(spins), dev(J))
        E, M = g.ising_energy()
        o = ea3d.Oracle(L, 1, synth.DYN_SEED, PHILOX)
        o.load_packed(spins, J)
        Eo, Mo = o.energy()
        assert (int(E[0]), int(M[0])) == (int(Eo[0]), int(Mo[0]))
        want.append((int(E[0]), int(M[0])))
        g.ising_destroy()
    assert want[0] != want[1]
    d_in = [(dev(s).flatten(), dev(J).flatten()) for s, J in inputs]
    E = torch.full((1,), 12345, dtype=torch.int64, device="cuda")
    M = torch.full((1,), 54321, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for k in (0, 1, 0, 0):     # two different calls in a row, then the first input again, twice
        binding.ising_energy_static(L, d_in[k][0], d_in[k][1], E, M)
        assert (int(E[0]), int(M[0])) == want[k], k
    binding.ising_energy_static(L, d_in[1][0], d_in[1][1], E)   # M not wanted
    assert int(E[0]) == want[1][0] and int(M[0]) == want[0][1]
    assert torch.cuda.memory_allocated() == before
    # back to back on one stream without a host synchronisation in between: stream order is enough
    E2 = torch.zeros(1, dtype=torch.int64, device="cuda")
    binding.ising_energy_static(L, d_in[0][0], d_in[0][1], E, M)
    binding.ising_energy_static(L, d_in[1][0], d_in[1][1], E2)
    torch.cuda.synchronize()
    assert int(E[0]) == want[0][0] and int(E2[0]) == want[1][0]
    # a handle of the same size working next to it is not disturbed, and does not disturb it
    g = Ising(L, 1, synth.DYN_SEED, PHILOX)
    g.ising_load_state(d_in[0][0].reshape(1, -1), d_in[0][1].reshape(1, 3, -1))
    g.ising_sweep(0.8, 2)
    binding.ising_energy_static(L, d_in[1][0], d_in[1][1], E, M)
    Eg, Mg = g.ising_energy()
    spins_now = g.ising_get_spins().flatten()
    binding.ising_energy_static(L, spins_now, d_in[0][1], E2)
    assert (int(E[0]), int(M[0])) == want[1] and int(E2[0]) == int(Eg[0])


@pytest.mark.gpu
def test_static_energy_rejects_sizes_beyond_its_scratch():
    L = 192
    spins, J = dev(synth.make_spins(L, 1, 1)).flatten(), dev(synth.make_couplings(L, 1, 2)).flatten()
    E = torch.zeros(1, dtype=torch.int64, device="cuda")
    with pytest.raises(binding.IsingError, match="ISING_STATIC_MAX_L"):
        binding.ising_energy_static(L, spins, J, E)
