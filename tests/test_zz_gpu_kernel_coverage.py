"""Runs last (file name): every tuned kernel instantiation the library holds must have been launched at least once by the
GPU tests before it -- the suite compares each launch with the oracle, so an instantiation missing here is one that no
parity test has run (VERDICT r1 "whole template families are never executed")."""
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def test_every_instantiation_was_launched_under_a_checker():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_09700_b200 import eri
    catalog, launched = set(eri.eri_kernel_catalog()), set(eri.eri_kernel_launched())
    if not any(x.startswith("coop 4 4 4 4") for x in launched):
        pytest.skip("run the whole GPU suite (pytest tests -m gpu): this check needs the other GPU tests in the same process")
    missing = sorted(catalog - launched)
    assert not missing, f"{len(missing)} of {len(catalog)} instantiations never launched: {missing[:20]}"
