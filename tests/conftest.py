import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


class Act:
    """Action-index layout of S:47: gather R | craft (1 or R) | buy R*P | sell R*P | noop."""

    def __init__(self, R, P, per_resource=False):
        self.R, self.P = R, P
        self.n_craft = R if per_resource else 1
        self.base_buy = R + self.n_craft
        self.base_sell = self.base_buy + R * P
        self.noop = self.base_sell + R * P
        self.A = self.noop + 1

    def gather(self, r):
        return r

    def craft(self, r=0):
        return self.R + (r if self.n_craft > 1 else 0)

    def buy(self, r, pidx):
        return self.base_buy + r * self.P + pidx

    def sell(self, r, pidx):
        return self.base_sell + r * self.P + pidx


@pytest.fixture
def small_params():
    from paper_2410_22165_b200 import inputs
    p = inputs.default_params()
    p.update(prices=list(range(1, 11)), tax_period=10, episode_length=50, rate_table=inputs.rate_table(11))
    return p
