"""CATAPULT oracle: plain CPU restatement of the paper's method.  TEST INFRASTRUCTURE ONLY."""
