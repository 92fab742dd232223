"""N > 1 host logic on CPU: two processes over `gloo` partition the frozen-phonon configurations and average
their outputs.  The per-configuration "output" is the oracle's PRISM result on a tiny case,
so the test also checks that the average over ranks equals the serial average."""
import os
import socket

import numpy as np
import pytest

from paper_1706_08563_b200 import sharding

torch = pytest.importorskip("torch")


def test_partition_covers_every_configuration_once():
    for n_ph in (1, 4, 8):
        for world in (1, 2, 3, 8):
            got = sorted(ph for r in range(world) for ph in sharding.phonons_for_rank(n_ph, world, r))
            assert got == list(range(max(n_ph, world)))
            sizes = [len(sharding.phonons_for_rank(n_ph, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        sharding.phonons_for_rank(4, 2, 2)


def _tiny_case():
    import oracle as O
    from helpers import oracle_params
    from paper_1706_08563_b200 import workloads as W
    w = W.scaled_test_case(32, 2, 2, 2, seed_index=41, density=0.2).with_(jitter=0.08, n_phonons=4)
    return O, w, oracle_params(w)


def _one_configuration(O, w, p, ph):
    lut_z, r_cut, lut_v = w.lut()
    v = O.potential(p, w.atoms_for_phonon(ph), w.z, lut_z, r_cut, lut_v)
    beams = O.beams(p)
    return O.prism_probes(p, O.smatrix(p, v, beams), beams, w.probe_xy())


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    O, w, p = _tiny_case()
    mine = sharding.phonons_for_rank(w.n_phonons, world, rank)
    acc = torch.zeros((w.n_probes, O.num_bins(p)), dtype=torch.float64)
    for ph in mine:
        acc += torch.from_numpy(_one_configuration(O, w, p, ph))
    sharding.phonon_average(acc, len(mine), dist)
    np.save(os.path.join(out_dir, f"rank{rank}.npy"), acc.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_average_equals_serial_average(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    O, w, p = _tiny_case()
    serial = np.mean([_one_configuration(O, w, p, ph) for ph in range(w.n_phonons)], axis=0)
    for r in range(2):
        got = np.load(tmp_path / f"rank{r}.npy")
        assert np.allclose(got, serial, rtol=1e-13, atol=1e-16)
    # configurations differ (the jitter is drawn per configuration), so the average is not a single run
    assert not np.allclose(serial, _one_configuration(O, w, p, 0), rtol=1e-6)


def test_single_process_average():
    acc = torch.full((3, 5), 6.0, dtype=torch.float64)
    sharding.phonon_average(acc, 3, None)
    assert torch.allclose(acc, torch.full((3, 5), 2.0, dtype=torch.float64))
