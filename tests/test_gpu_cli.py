"""-m gpu: the command-line entry (paper_1005_5198_b200.cli) makes the same map as the oracle for a lens file."""
import numpy as np
import pytest

from oracle import oracle
from paper_1005_5198_b200 import cli

pytestmark = pytest.mark.gpu


def test_cli_writes_the_oracles_map(tmp_path, capsys):
    args = (0.4, 1.0, 0.1, 64, 36.0, 8.0)
    g = oracle.geometry(*args)
    xy = np.random.default_rng(8).uniform(-g.r_star / 2, g.r_star / 2, size=(40, 2))
    mass = np.random.default_rng(9).uniform(0.5, 2.0, size=40)
    np.savetxt(tmp_path / "lenses.txt", xy, fmt="%.17g")
    np.savetxt(tmp_path / "masses.txt", mass, fmt="%.17g")
    rc = cli.main(["--sigma", "0.4", "--gamma", "0.1", "--n-pix", "64", "--n-rays", "36", "--L", "8",
                   "--lenses", str(tmp_path / "lenses.txt"), "--masses", str(tmp_path / "masses.txt"),
                   "--precision", "fp64", "--out", str(tmp_path / "map.npy"), "--pgm", str(tmp_path / "map.pgm")])
    assert rc == 0
    counts = np.load(tmp_path / "map.npy")
    omap, ost = oracle.shoot(*args, xy, mass=mass)
    assert counts.dtype == np.uint32 and (counts != omap).sum() <= 2 and abs(int(counts.sum()) - ost["rays_in_map"]) <= 2
    pgm = (tmp_path / "map.pgm").read_bytes()
    assert pgm.startswith(b"P5\n64 64\n255\n") and len(pgm) == len(b"P5\n64 64\n255\n") + 64 * 64
    out = capsys.readouterr().out
    assert "lenses 40" in out and "interactions/s" in out
    # synthetic disk + random rays path
    assert cli.main(["--sigma", "0.4", "--n-pix", "32", "--n-rays", "16", "--L", "4", "--seed", "3", "--random-rays", "5",
                     "--dm-hist", "6"]) == 0
    hist = [ln for ln in capsys.readouterr().out.splitlines() if ln.startswith("dm [")]
    assert len(hist) == 6 and 0 < sum(int(ln.split()[-1]) for ln in hist) <= 32 * 32
