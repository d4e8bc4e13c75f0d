"""no_hf_energy_static: the Hartree-Fock energy for callers that must not allocate GPU memory.

Why the entry point exists: the library is meant to be driven by many integration workers that share one GPU
(PAPER.md:182-186).  A cudaMalloc / cudaFree issued by one of them is a device-wide event that stalls the others, a
host program that gave all of HBM to its own pool gets out-of-memory from any later cudaMalloc, and some codes forbid
allocation after start-up altogether.  no_hf_energy grows a cudaMalloc arena on demand; no_hf_energy_static keeps the
same intermediates in a fixed 7.25 MiB `static __device__` array inside libno3n.so and rejects grids beyond 4096
nodes with NO_ERR_LIMIT.

What is checked: the new entry point against the EXISTING path (no_hf_energy, itself checked against the oracle in
test_parity_gpu.py) at the tolerance those tests use for the energy (relative 1e-11), on two calls in a row that
share the array: a large multi-pass call first, so that the second, small one runs over the first one's leftovers
(a missing clear of the accumulator, or a read of stale configurations, fails the second comparison), then the first
again.  Also the limit and the error text.

This file is named so that pytest collects it last (`pytest --collect-only`): under `-x` a failure here cannot hide
the parity tests.  It holds no state of its own, so it passes alone in a fresh process and after the other files."""
import pytest

torch = pytest.importorskip("torch")

from paper_2603_24532_b200 import NormalOrdering, binding, build   # noqa: E402

pytestmark = pytest.mark.gpu

REL_TOL = 1e-11          # tolerance of the Hartree-Fock energy in tests/test_parity_gpu.py
PHYS = dict(c1=-0.81, c3=-3.2, c4=5.4, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0,
            Lambda=500.0, n_reg=4)


@pytest.fixture(scope="module", autouse=True)
def _built():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    build.build()
    binding.load()


def test_static_scratch_energy_equals_the_allocating_path_on_two_calls_in_a_row():
    big = NormalOrdering(device=0, kf_n=1.4, kf_p=1.0, n_r=5, n_cos=4, n_phi=6, **PHYS)    # two spheres: four pair grids
    small = NormalOrdering(device=0, kf_n=1.1, kf_p=1.1, n_r=3, n_cos=3, n_phi=2, **PHYS)  # one shared pair grid
    try:
        # reference values from the existing, allocating path
        want_big = big.hf_energy(7, 7, 6)         # 294 nodes -> 86436 pairs: two passes of the static path (65536 + 20900)
        want_small = small.hf_energy(2, 3, 2)     # 12 nodes -> 144 pairs: a corner of the array the big call filled
        assert abs(want_big) > 1e-8 and abs(want_small) > 1e-8
        # two calls in a row on the shared array, then the first once more over the second one's leftovers
        got_big = big.hf_energy_static(7, 7, 6)
        got_small = small.hf_energy_static(2, 3, 2)
        again_big = big.hf_energy_static(7, 7, 6)
        assert got_big == pytest.approx(want_big, rel=REL_TOL)
        assert got_small == pytest.approx(want_small, rel=REL_TOL)
        assert again_big == got_big               # fixed summation order and no dependence on what the array held
        # a small grid is one pass in both paths: same kernels, same order, same bits
        assert got_small == want_small
        # the other kernel layout (one CTA per configuration) through the same array
        binding.no_set_layout(small._h, 2)
        assert small.hf_energy_static(2, 3, 2) == pytest.approx(small.hf_energy(2, 3, 2), rel=REL_TOL)
    finally:
        big.close()
        small.close()


def test_static_scratch_rejects_grids_beyond_its_capacity_without_touching_the_gpu():
    no = NormalOrdering(device=0, kf_n=1.0, kf_p=0.0, n_r=2, n_cos=2, n_phi=2, **PHYS)
    try:
        with pytest.raises(binding.NoError) as err:
            no.hf_energy_static(17, 16, 16)       # 4352 nodes > NO_HF_STATIC_MAX_NODES
        assert err.value.code == binding.NO_ERR_LIMIT
        assert "capacity" in str(err.value)
        # the largest grid that fits is accepted: 4096^2 pairs, 256 passes through the array
        e = no.hf_energy_static(16, 16, 16)
        assert e == pytest.approx(no.hf_energy(16, 16, 16), rel=REL_TOL)
    finally:
        no.close()
