"""CPU: the host-side bookkeeping the benchmark relies on -- roofline arithmetic, the seeded input
recipes and the batch-order tables.  No GPU, no oracle."""
import numpy as np
import pytest

from paper_2606_30497_b200 import datagen, roofline


def test_f_step_matches_the_survey_table():
    # F_step = 4BIH + 5BH + 2B + 2(IH + H); the paper's MAC counts are half of the products
    assert roofline.f_step(256, 256) == 8_733_696
    assert roofline.f_step(256, 64) == 2_183_808
    assert roofline.f_step(256, 1024) == 34_933_248
    assert roofline.f_step(32, 256) == 1_106_496
    assert roofline.f_step(4096, 256) == 139_485_696
    macs = 2 * 256 * 32 * 256 + 3 * 256 * 256          # eqs. 1, 8 + eqs. 3, 6, 7 (4,390,912)
    assert macs == 4_390_912


def test_floors_match_the_survey_table():
    assert roofline.train_floor_us(256, 256, 8, 1965.0) == pytest.approx(2.170, abs=1e-3)
    assert roofline.train_floor_us(256, 256, 16, 1965.0) == pytest.approx(1.085, abs=1e-3)
    assert roofline.train_floor_us(4096, 256, 8, 1965.0) == pytest.approx(34.66, abs=1e-2)
    assert roofline.eval_bytes_per_sample() == 132 and roofline.eval_flop_per_sample(256) == 16_899
    assert roofline.step_bytes(256) == 33_792
    # the tensor-core variant's floor is far below the exact kernel's and ordered BF16 < TF32
    for h in (32, 64, 128, 256, 512, 1024):
        tf, bf = roofline.tc_train_floor_us(256, h, 1965.0, False), roofline.tc_train_floor_us(256, h, 1965.0, True)
        assert 0 < bf < tf < roofline.train_floor_us(256, h, roofline.tc_train_cluster(h), 1965.0)


def test_configs_are_the_baseline_json_ones():
    c = datagen.CONFIGS
    assert (c["config1"].n, c["config1"].batch, c["config1"].epochs, c["config1"].shuffle) == (1024, 256, 1, False)
    assert (c["config2"].n, c["config2"].epochs, c["config3"].n, c["config3"].epochs) == (65536, 10, 1048576, 10)
    assert [m.hidden for m in datagen.sweep("config4")] == [64, 128, 512, 1024]
    assert [m.batch for m in datagen.sweep("config5")] == [32, 256, 1024, 4096]
    assert all(m.n == 4194304 and m.epochs == 3 for m in datagen.sweep("config5"))


def test_dataset_recipe_is_seeded_and_prefix_stable():
    X, Y = datagen.make_dataset(4096, 0.1)
    X2, Y2 = datagen.make_dataset(1024, 0.1)
    assert X.dtype == np.float32 and Y.dtype == np.float32 and X.shape == (4096, 32) and Y.shape == (4096,)
    assert np.array_equal(X[:1024], X2)                 # configs 2-4 are leading rows of config 5's matrix (bench.py relies on it)
    assert np.array_equal(Y[:1024], Y2)
    assert abs(float(X.mean())) < 0.02 and abs(float(X.var()) - 1.0) < 0.03
    assert 0.25 < float(Y.var()) < 0.42                 # var(Y) ~ 0.33


@pytest.mark.parametrize("n,batch,epochs", [(1024, 256, 3), (1000, 256, 2), (7, 1, 2), (3000, 5000, 2)])
def test_order_tables_are_per_epoch_permutations(n, batch, epochs):
    nb = datagen.num_batches(n, batch)
    o = datagen.make_order(n, batch, epochs, True)
    assert o.shape == (epochs, nb) and o.dtype == np.int32
    for e in range(epochs):
        assert sorted(o[e].tolist()) == list(range(nb))
    s = datagen.make_order(n, batch, epochs, False)
    assert all(s[e].tolist() == list(range(nb)) for e in range(epochs))
    assert np.array_equal(o, datagen.make_order(n, batch, epochs, True))      # seeded
