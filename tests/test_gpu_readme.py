"""The usage example printed in README.md runs as written."""
import os
import re

import pytest

pytestmark = pytest.mark.gpu


def test_readme_example_runs(repo_root):
    text = open(os.path.join(repo_root, "README.md")).read()
    blocks = re.findall(r"```python\n(.*?)```", text, flags=re.S)
    assert len(blocks) == 1
    ns = {}
    exec(compile(blocks[0], "README.md", "exec"), ns)
    assert tuple(ns["y"].shape) == (32, 100000) and tuple(ns["xa"].shape) == (32, 256, 256)
    assert tuple(ns["xs"].shape) == (32, 256, 256) and tuple(ns["xr"].shape) == (256, 256)
    assert bool(ns["xr"].isfinite().all())
