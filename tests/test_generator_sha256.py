"""The seeded generator is the one thing the oracle and the CUDA path share (it holds none of the method's arithmetic):
its output must not drift.  The digests below were written by `python -m emu_synth.sha256`."""
from emu_synth.sha256 import batch_digest, config_digest

EXPECTED = {
    0: (1721, "058ccaab44d15c3d56fb5b6585abea4f4cf543acd1c8a8f1cf1afa594c899f3e"),
    1: (23400, "d4ff2f9c77a705abd00a72f1f58a5a4377b766d3d470d5b26b36ecf32db7d6e9"),
    2: (24024, "421428ea464d3bf9e713d688fd83e12666e74dfd323f8ab4b4ba84f96fd67ad5"),
    3: (27915, "0f7984738e69ef855f4a60f6b50e8a4ca6a08990d588eaa744274e162b8df580"),
}


def test_configs_0_to_3():
    for c, want in EXPECTED.items():
        assert config_digest(c) == want, c


def test_first_views_of_the_throughput_batch():
    assert batch_digest(0, 16) == (1025119, "bf0e4f4aa4bdf620508074a790481f68e26add1e151bb242b912c7b5db214505")
