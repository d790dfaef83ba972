"""CPU oracle for the PIMC hot path -- TEST INFRASTRUCTURE ONLY (see pimc_oracle.cpp)."""
from .oracle import OracleChain, philox4x32_10, philox_bulk, draw_words, u01_from_word, u01_from_two_words, \
    u01f_from_word, box_muller, step_increment, rhs, model_np, lib  # noqa: F401
