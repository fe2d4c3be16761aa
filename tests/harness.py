"""Test harness = the oracle-side world builders (``oracle/worlds.py``: seeded synthetic state of a config, planned and
placed by the oracle).  Kept under this name for the tests; ``bench.py``'s oracle legs import ``oracle.worlds`` directly."""
from oracle.worlds import *  # noqa: F401,F403
from oracle.worlds import GUARD, OracleSide, Step, ParamWorld, KVWorld  # noqa: F401
