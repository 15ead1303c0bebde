#!/bin/sh
# Builds the oracle (test infrastructure) into oracle/librc_oracle.so.
set -e
cd "$(dirname "$0")"
g++ -std=c++17 -O2 -fPIC -shared -Wall -Wextra -o librc_oracle.so rc_oracle.cpp
