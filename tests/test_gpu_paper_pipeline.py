"""The paper's own labelling pipeline as an ablation baseline (sw_label_paper): self-labelling on B x B
tiles + label relaxation / hierarchical sewing must give the canonical labelling of the oracle, bit for bit (-m gpu)."""
import math

import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import binding, inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (the product has no CPU path)")
    binding.lib()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def paper_case(L, codes, methods=(0, 1), Bs=(8, 16, 32)):
    want, nc = oracle.label(L, codes)
    lat = binding.Lattice(L, 2, 0.1, 0)
    packed = dev(inputs.pack_codes(codes))
    out = torch.empty(L * L, dtype=torch.int32, device="cuda")
    for method in methods:
        for B in Bs:
            if L % B or (method == 1 and (L // B) & (L // B - 1)):
                continue
            out.fill_(-7)
            st = lat.label_paper(method, B, packed, out)
            got = out.cpu().numpy()
            assert np.array_equal(got, want), f"L={L} method={method} B={B}: {int((got != want).sum())} labels differ"
            assert lat.observables(spins=False, clusters=False)["n_clusters"] == nc
            assert 1 <= st["selflabel_passes_max"] <= B * B
            if method == 0:
                assert st["relax_iterations"] >= 1 and st["sewing_levels"] == 0 and st["ms_wrap"] == 0.0
            else:
                assert st["sewing_levels"] == int(math.log2(L // B)) and st["relax_iterations"] == 0
                assert 0.0 < st["ms_wrap"] <= st["ms_consolidate"]          # the wrap-around step is timed on its own
    lat.close()


@pytest.mark.parametrize("L", [32, 64, 96, 256, 512])
@pytest.mark.parametrize("p", [0.3, 0.5, 0.62])
def test_random_bonds(L, p):
    paper_case(L, inputs.random_bond_codes(L, p, p, 100 + L))


def test_structured_bond_sets():
    for L in (32, 128):
        N = L * L
        paper_case(L, np.zeros(N, np.uint8))
        paper_case(L, np.full(N, 3, np.uint8))
        paper_case(L, np.full(N, 1, np.uint8))
        paper_case(L, np.full(N, 2, np.uint8))
        paper_case(L, inputs.snake_codes(L))
        paper_case(L, inputs.spiral_codes(L))
        c = np.zeros(N, np.uint8); c[L - 1] = 1; c[(L - 1) * L] |= 2        # one wrap bond per direction
        paper_case(L, c)


def test_critical_sw_bonds_L1024_and_relaxation_count():
    """Bonds of an equilibrated critical configuration: clusters span many tiles.  n_relax grows with L/B (Eq. 13)."""
    L, seed = 1024, 5
    lat = binding.Lattice(L, 2, oracle.beta_c(2), seed, with_bonds=True)
    lat.init_spins(1)
    lat.sweep(60)
    lat.activate()
    codes = inputs.unpack_codes(lat.bonds.cpu().numpy())
    want, nc = oracle.label(L, codes)
    out = torch.empty(L * L, dtype=torch.int32, device="cuda")
    its = {}
    for B in (8, 32):
        st = lat.label_paper(0, B, None, out)
        assert np.array_equal(out.cpu().numpy(), want)
        its[B] = st["relax_iterations"]
        st = lat.label_paper(1, B, None, out)
        assert np.array_equal(out.cpu().numpy(), want)
    assert its[8] > its[32] > 3
    lat.close()


def test_bad_arguments():
    lat = binding.Lattice(96, 2, 0.1, 0, with_bonds=True)
    for method, B in ((2, 16), (0, 12), (0, 64), (1, 32)):             # 96 / 32 = 3 tiles: not a power of two for sewing
        with pytest.raises(binding.SwError):
            lat.label_paper(method, B)
    lat.close()
