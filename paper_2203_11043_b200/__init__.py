"""gcoreccd-b200: B200-native (sm_100a) hot path of the G-CoReCCD charge-transport simulator.

Importing the package is cheap and loads no native code; `paper_2203_11043_b200.binding`
loads the C-ABI library (include/gcoreccd.h) on first use and fails loudly if it is missing.
"""
__all__ = ["binding", "build"]
